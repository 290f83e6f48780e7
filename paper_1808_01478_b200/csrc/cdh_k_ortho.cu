// Tile kernels of the orthorhombic box, one per form of the rint (cdh_variants.h, cdh_fast.cuh).
#include "cdh_math32.cuh"
#include "cdh_variants.cuh"
namespace cdh {
Variant fast_variant_ortho(int form, int mode, int shape) {
    if (form == ORTHO_FUSED) return shapes_of<MathFast<BOX_ORTHO, ORTHO_FUSED>, CDH_MINB, CDH_BIG_T_PERIODIC, true, CDH_HYB_T_ORTHO>(mode, shape);
    if (form == ORTHO_EXACT) return shapes_of<MathFast<BOX_ORTHO, ORTHO_EXACT>, CDH_MINB, CDH_BIG_T_PERIODIC, true, CDH_HYB_T_ORTHO>(mode, shape);
    return shapes_of<MathFast<BOX_ORTHO, ORTHO_PLAIN>, CDH_MINB, CDH_BIG_T_PERIODIC, true, CDH_HYB_T_ORTHO>(mode, shape);
}
}
