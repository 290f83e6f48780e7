// The cross-validation tile kernels: the pinned sequence spelled with IEEE intrinsics, and the two aggregation variants of
// its histogram update (cdh_variants.h, cdh_kernels.cuh).  Bin-range split and global mode only.
#include "cdh_math32.cuh"
#include "cdh_variants.cuh"
namespace cdh {
template <int VAR>
static Variant simple_of(int box, int mode, int shape) {
    if (box == BOX_NONE) return shapes_of<MathSimple<BOX_NONE, VAR>, 2, CDH_BIG_T, false>(mode, shape);
    if (box == BOX_ORTHO) return shapes_of<MathSimple<BOX_ORTHO, VAR>, 2, CDH_BIG_T_PERIODIC, false, CDH_HYB_T_ORTHO>(mode, shape);
    return shapes_of<MathSimple<BOX_TRI, VAR>, 2, CDH_BIG_T_PERIODIC, false>(mode, shape);
}
Variant simple_variant(int box, int var, int mode, int shape) {
    if (var == VAR_SIMPLE_MATCH && mode == MODE_SPLIT) return simple_of<VAR_SIMPLE_MATCH>(box, mode, shape);
    if (var == VAR_SIMPLE_PLAIN && mode == MODE_SPLIT) return simple_of<VAR_SIMPLE_PLAIN>(box, mode, shape);
    return simple_of<VAR_SIMPLE>(box, mode, shape);
}
}
