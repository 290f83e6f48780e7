// cdh_variants.h -- the table of tile-kernel instantiations (host side).  The kernels are instantiated in several
// translation units (cdh_k_*.cu) so that the library builds in parallel; cdh_api.cu picks one per launch.
#pragma once
#include <cstdint>

namespace cdh {

struct Variant {
    const void* fn;     // __global__ function: launched with cudaLaunchKernel, one argument (TileParams / TileParams64)
    int threads;        // CTA size
};

// CTA shapes: 256 threads with several CTAs per SM; one big CTA per SM (1024 threads, 512 in double) when the private
// histogram leaves room for one CTA only; 256 threads with the small-species SKIP form (cdh_sched.cuh).
enum Shape { SHAPE_256 = 0, SHAPE_BIG = 1, SHAPE_256_SKIP = 2 };

// form: 0 for BOX_NONE; ORTHO_PLAIN / ORTHO_FUSED / ORTHO_EXACT for BOX_ORTHO; TRI_GENERAL / TRI_UPPER / TRI_UPPER_B01,
// optionally | TRI_WIDE, or TRI_GENERAL | TRI_NOPRUNE (| TRI_WIDE) for BOX_TRI.  Returns {nullptr, 0} for a combination
// that is not built.
Variant fast_variant_none(int mode, int shape);
Variant fast_variant_ortho(int form, int mode, int shape);
Variant fast_variant_tri(int form, int mode, int shape);          // narrow range (n_k in {-1, 0, 1})
Variant fast_variant_tri_wide(int form, int mode, int shape);     // TRI_WIDE forms
Variant simple_variant(int box, int var, int mode, int shape);    // var: VAR_SIMPLE / VAR_SIMPLE_MATCH / VAR_SIMPLE_PLAIN
Variant f64_variant(int box, bool pbox, int mode, int shape);

}  // namespace cdh
