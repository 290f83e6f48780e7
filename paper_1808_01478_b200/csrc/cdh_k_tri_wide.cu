// Tile kernels of the triclinic box for coordinates spanning up to 64 cells (TRI_WIDE; cdh_variants.h, cdh_fast.cuh).
#include "cdh_math32.cuh"
#include "cdh_variants.cuh"
namespace cdh {
Variant fast_variant_tri_wide(int form, int mode, int shape) {
    if (form == (TRI_UPPER_B01 | TRI_WIDE)) return shapes_of<MathFast<BOX_TRI, TRI_UPPER_B01 | TRI_WIDE>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == (TRI_UPPER | TRI_WIDE)) return shapes_of<MathFast<BOX_TRI, TRI_UPPER | TRI_WIDE>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == (TRI_GENERAL | TRI_WIDE | TRI_NOPRUNE)) return shapes_of<MathFast<BOX_TRI, TRI_GENERAL | TRI_WIDE | TRI_NOPRUNE>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    if (form == (TRI_GENERAL | TRI_WIDE)) return shapes_of<MathFast<BOX_TRI, TRI_GENERAL | TRI_WIDE>, 2, CDH_BIG_T_PERIODIC>(mode, shape);
    return {nullptr, 0};
}
}
