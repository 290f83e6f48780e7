// cdh_variants.cuh -- instantiates the launch shapes of one arithmetic policy (included by the cdh_k_*.cu units).
#pragma once
#include "cdh_variants.h"
#include "cdh_sched.cuh"

#ifndef CDH_MINB
#define CDH_MINB 3      // resident CTAs per SM the 256-thread NONE / ORTHO fast variants are register-bounded for
                        // (80 registers; measured +1.5 % over 2; the triclinic variants need 128 registers: 2)
#endif
#ifndef CDH_BIG_T_PERIODIC
#define CDH_BIG_T_PERIODIC 512  // ... of the packed-fp32 kernels for periodic boxes: they need 72-128 registers, and the 64 a 1,024-thread
                                // CTA leaves them cost more than its 32 warps bring (100,000 points, 20,000-50,000 bins, 1,024 -> 512
                                // threads: orthorhombic 1,304 -> 1,351, triclinic 734-695 -> 780-807 Gpairs/s)
#endif
#ifndef CDH_HYB_T_ORTHO
#define CDH_HYB_T_ORTHO 1024    // hybrid mode hides the latency of its L2 reductions with warps: orthorhombic, 100,000 bins: 840 with 1,024
                                // threads, 763 with 512 (triclinic: 556 against 578, so it keeps 512)
#endif
#ifndef CDH_BIG_T
#define CDH_BIG_T 1024  // threads of the one-CTA-per-SM variants (32 warps/SM: config 5 +5 % over 512)
#endif

namespace cdh {

// MINB: resident CTAs per SM the 256-thread kernels are register-bounded for; BIG_T: threads of the one-CTA-per-SM shape;
// HYB_T: threads of the hybrid-mode kernels.  All launches of a plan share one i-tile size (the work tables are built for it), so
// the fast and the cross-validation kernels of a box type must be given the same BIG_T and HYB_T.
// FULL = false builds only what the cross-validation variants need (bin-range split and global mode).
template <class M, int MINB, int BIG_T, bool FULL = true, int HYB_T = BIG_T>
Variant shapes_of(int mode, int shape) {
    if constexpr (FULL) {
        if (mode == MODE_SHARED) {
            if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_SHARED, false>, BIG_T};
            if (shape == SHAPE_256_SKIP) return {(const void*)tile_kernel<M, 256, MINB, MODE_SHARED, true>, 256};
            return {(const void*)tile_kernel<M, 256, MINB, MODE_SHARED, false>, 256};
        }
        if (mode == MODE_HYBRID) return {(const void*)tile_kernel<M, HYB_T, 1, MODE_HYBRID, false>, HYB_T};
    }
    if (mode == MODE_SPLIT) {
        if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, BIG_T, 1, MODE_SPLIT, false>, BIG_T};
        return {(const void*)tile_kernel<M, 256, MINB, MODE_SPLIT, false>, 256};
    }
    if (mode == MODE_GLOBAL) {
        // the big shape only for the cross-validation kernels: they are the out-of-range fallback of MODE_HYBRID plans, whose
        // work tables are built for the big i-tile
        if constexpr (!FULL) if (shape == SHAPE_BIG) return {(const void*)tile_kernel<M, HYB_T, 1, MODE_GLOBAL, false>, HYB_T};
        return {(const void*)tile_kernel<M, 256, MINB, MODE_GLOBAL, false>, 256};
    }
    return {nullptr, 0};
}

}  // namespace cdh
