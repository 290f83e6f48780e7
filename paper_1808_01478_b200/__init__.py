"""paper_1808_01478_b200 -- B200-native particle-pair distance histograms (CADISHI hot path).

The product is ``libcdh.so`` (C ABI in ``include/cdh.h``, CUDA kernels in ``csrc/``); this package is
its thin Python binding plus the seeded input generators (``inputs``).  Importing the package does not
load the library; the first call does, and fails loudly if it was not built.
"""
from . import inputs  # noqa: F401
from .binding import (BOX_NONE, BOX_ORTHO, BOX_TRICLINIC, F32, F64, FLAG_MAX_SMEM_BINS_SHIFT,  # noqa: F401
                      FLAG_ACCUMULATE, FLAG_GLOBAL_HIST, FLAG_NO_AGGREGATE, FLAG_NO_ITEM_TABLE, FLAG_NO_PDL, FLAG_NO_PRUNE, FLAG_SIMPLE_KERNEL, FLAG_TIME_KERNELS, FLAG_WARP_AGGREGATE, CdhError,
                      Context, cdh_bench_dsmem_atomics, cdh_bench_fp32_rate, cdh_bench_inner_loop, cdh_bench_shared_atomics, cdh_create, cdh_histograms_noalloc, NOALLOC_MAX_BINS, NOALLOC_MAX_PADDED_PARTICLES, cdh_selftest_sqrt, cdh_selftest_sqrt_f64,
                      cdh_strerror, load)


def histograms_device(ctx: "Context", problem, stream=None, precision: int = F32):
    """Run ``cdh_histograms`` on an ``inputs.Problem``: copies the coordinates to the context's device
    with torch (plumbing), calls the library, returns a torch uint64-as-int64 CUDA tensor [n_hist, n_bins]
    (not synchronised).  ``precision=F64`` widens the float32 coordinates to double first (exact)."""
    import numpy as np
    import torch
    dev = torch.device("cuda", ctx.device)
    host = problem.coords.astype(np.float64) if precision == F64 else problem.coords
    coords = torch.from_numpy(host).to(dev)
    out = torch.empty((problem.n_hist, problem.n_bins), dtype=torch.int64, device=dev)
    if stream is not None and hasattr(stream, "cuda_stream"):
        # coords was filled on torch's current stream and is read on `stream`: order the two, and keep the caching allocator
        # from handing the block to someone else before the repack kernel has read it (coords is dropped on return)
        stream.wait_stream(torch.cuda.current_stream(dev))
        coords.record_stream(stream)
        out.record_stream(stream)
    ctx.cdh_histograms(coords, problem.n_frames, problem.species_offsets, problem.box_type, problem.box,
                       problem.r_max, problem.n_bins, out, precision=precision, stream=stream)
    return out
