// The double-precision tile kernels (cdh_variants.h, cdh_f64.cuh).
#include "cdh_f64.cuh"
#include "cdh_variants.cuh"
namespace cdh {
Variant f64_variant(int box, bool pbox, int mode, int shape) {
    if (box == BOX_NONE) return shapes_of<MathF64<BOX_NONE, false>, 2, 512>(mode, shape);
    if (box == BOX_ORTHO) return shapes_of<MathF64<BOX_ORTHO, false>, 2, 512>(mode, shape);
    if (pbox) return shapes_of<MathF64<BOX_TRI, true>, 2, 512>(mode, shape);
    return shapes_of<MathF64<BOX_TRI, false>, 2, 512>(mode, shape);
}
}
