// cdh_variants.cuh -- instantiates the launch shapes of one arithmetic policy (included by the cdh_k_*.cu units).
#pragma once
#include "cdh_variants.h"
#include "cdh_sched.cuh"

#ifndef CDH_MINB
#define CDH_MINB 3      // resident CTAs per SM the 256-thread NONE / ORTHO fast variants are register-bounded for
                        // (80 registers; measured +1.5 % over 2; the triclinic variants need 128 registers: 2)
#endif
#ifndef CDH_BIG_T
#define CDH_BIG_T 1024  // threads of the one-CTA-per-SM variants (32 warps/SM: config 5 +5 % over 512)
#endif

namespace cdh {

// MINB: resident CTAs per SM the 256-thread kernels are register-bounded for; BIG_T: threads of the one-CTA-per-SM shape.
// FULL = false builds only what the cross-validation variants need (bin-range split and global mode).
template <class M, int MINB, int BIG_T, bool FULL = true>
Variant shapes_of(int mode, int shape) {
    if constexpr (FULL) {
        if (mode == MODE_SHARED) {
            if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_SHARED, false>, BIG_T};
            if (shape == SHAPE_256_SKIP) return {(const void*)tile_kernel<M, 256, MINB, MODE_SHARED, true>, 256};
            return {(const void*)tile_kernel<M, 256, MINB, MODE_SHARED, false>, 256};
        }
        if (mode == MODE_HYBRID) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_HYBRID, false>, BIG_T};
    }
    if (mode == MODE_SPLIT) {
        if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_SPLIT, false>, BIG_T};
        return {(const void*)tile_kernel<M, 256, MINB, MODE_SPLIT, false>, 256};
    }
    if (mode == MODE_GLOBAL) {
        // the big shape only for the cross-validation kernels: they are the out-of-range fallback of MODE_HYBRID plans, whose
        // work tables are built for the big i-tile
        if constexpr (!FULL) if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_GLOBAL, false>, BIG_T};
        return {(const void*)tile_kernel<M, 256, MINB, MODE_GLOBAL, false>, 256};
    }
    return {nullptr, 0};
}

}  // namespace cdh
