// Tile kernels without a box (cdh_variants.h).
#include "cdh_math32.cuh"
#include "cdh_variants.cuh"
namespace cdh {
Variant fast_variant_none(int mode, int shape) { return shapes_of<MathFast<BOX_NONE, 0>, CDH_MINB, CDH_BIG_T>(mode, shape); }
}
