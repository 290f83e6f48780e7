// Tile kernels of the triclinic box, fractional range <= 1.49 (cdh_variants.h, cdh_fast.cuh).
#include "cdh_math32.cuh"
#include "cdh_variants.cuh"
namespace cdh {
Variant fast_variant_tri(int form, int mode, int shape) {
    if (form == TRI_UPPER_B01) return shapes_of<MathFast<BOX_TRI, TRI_UPPER_B01>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == TRI_UPPER) return shapes_of<MathFast<BOX_TRI, TRI_UPPER>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == (TRI_GENERAL | TRI_NOPRUNE)) return shapes_of<MathFast<BOX_TRI, TRI_GENERAL | TRI_NOPRUNE>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == TRI_GENERAL) return shapes_of<MathFast<BOX_TRI, TRI_GENERAL>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    return {nullptr, 0};
}
}
