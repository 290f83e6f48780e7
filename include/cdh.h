/*
 * cdh.h -- C ABI of the B200-native particle-pair distance histogram library (libcdh.so).
 *
 * What the library computes is the hot path of Reuter & Koefinger, "CADISHI" (arxiv 1808.01478;
 * citations are PAPER.md:<line> of /root/reference/PAPER.md):
 *   - Algorithm 1 (section 2.2): for every particle i of species p and j of species q,
 *     distance vector, minimum image (periodic boxes), r = sqrt(x^2+y^2+z^2),
 *     kappa = (int) n_bins * r / r_max, ++hist[kappa];
 *   - one species (p == q): unique pairs j > i only, N(N-1)/2 of them;
 *   - half-open bins r_kappa <= r < r_kappa + dr (Eq. 4);
 *   - minimum image dx' = dx - b nint(b^-1 dx) (Eq. 5); b diagonal for an
 *     orthorhombic box; for a triclinic box dx' is additionally shifted to the 26
 *     neighbouring cells and the minimum taken (section 2.3);
 *   - one call takes the whole contiguous multi-species coordinate set and returns ALL species-pair
 *     histograms; counts are 32 bit inside the kernels and 64 bit in the result
 *     (PAPER.md:161, 205); histograms of all frames of the call are summed (Eq. 2);
 *   - device scratch is allocated at the first call and reused.
 * The per-pair IEEE-754 operation sequence ("pinned sequence") the integers are defined by is stated
 * in DESIGN.md; the kernels reproduce it bit for bit.
 *
 * Threading: one context per device, not thread-safe; a context must not be used on two streams
 * concurrently.  No call prints, throws or aborts.
 */
#ifndef CDH_H
#define CDH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* box_type */
#define CDH_BOX_NONE       0   /* no periodic box */
#define CDH_BOX_ORTHO      1   /* orthorhombic periodic box (b diagonal) */
#define CDH_BOX_TRICLINIC  2   /* general triclinic periodic box (Eq. 5 + neighbour shift) */

/* precision */
#define CDH_F32 0              /* the pinned fp32 sequence (built) */
#define CDH_F64 1              /* the same sequence in double (coords are doubles); plain IEEE arithmetic,
                                  no packed / magic-number shortcuts */

/* return codes */
#define CDH_OK                 0
#define CDH_ERR_INVALID_ARG  (-1)  /* detected before anything is enqueued; out untouched */
#define CDH_ERR_UNSUPPORTED  (-2)  /* the library was built without the kernel variant the call needs (nothing enqueued) */
#define CDH_ERR_ALLOC        (-3)  /* device or pinned-host allocation failed */
#define CDH_ERR_CUDA         (-4)  /* a CUDA runtime call failed; text via cdh_last_error() */

/* cdh_create flags: 0 for production.  The other bits force a kernel variant (tests, ncu A/B runs);
 * every variant returns the same integers. */
#define CDH_FLAG_SIMPLE_KERNEL   (1u << 0) /* plain scalar kernel with library sqrtf/rintf/floorf: the
                                              cross-validation kernel */
#define CDH_FLAG_NO_PRUNE        (1u << 1) /* triclinic: always search the 27 shifts */
#define CDH_FLAG_WARP_AGGREGATE  (1u << 2) /* plain kernel, equal bins of a warp aggregated in software
                                              (__match_any_sync, one ATOMS.ADD per distinct bin) */
#define CDH_FLAG_NO_AGGREGATE    (1u << 3) /* plain kernel, one ATOMS.ADD per lane (no aggregation at all);
                                              production uses ATOMS.POPC.INC, which merges equal addresses in hardware */
#define CDH_FLAG_TIME_KERNELS     (1u << 4) /* record CUDA events around the tile kernel(s) of every call
                                              (measurement; read with cdh_call_kernel_ms) */
#define CDH_FLAG_GLOBAL_HIST      (1u << 5) /* no private histogram: every kept pair adds to the uint64 result
                                              directly (chosen automatically beyond 16 shared-memory windows of bins;
                                              between one and 16 windows the library keeps the most populated window of
                                              every histogram row in shared memory and sends the rest to L2, in one sweep) */
#define CDH_FLAG_ACCUMULATE       (1u << 6) /* cdh_histograms ADDS to `out` instead of overwriting it: a caller can feed a
                                              trajectory in chunks of frames (the paper's writer sums every 100 frames,
                                              PAPER.md:338).  Not for cdh_histograms_host (its device result is scratch) */
#define CDH_FLAG_NO_PDL           (1u << 7) /* launch the tile kernels without programmatic stream serialization (A/B of the
                                              small-call latency: by default a tile launch starts its prologue while the
                                              kernel before it still runs and waits on the device before it reads its data) */
#define CDH_FLAG_NO_ITEM_TABLE    (1u << 8) /* build no per-item descriptor table: the kernel looks every work item up in the
                                              row / segment tables, as calls with more than 262,144 items do (tests) */
#define CDH_FLAG_MAX_SMEM_BINS_SHIFT 12    /* bits 12..31: if non-zero, cap on the bins one CTA keeps in
                                              shared memory (forces the bin-range-split path) */

typedef struct cdh_ctx cdh_ctx;  /* opaque; owns device scratch (repacked coordinates, work tables) only */

/* Create a context on CUDA device `device` (HOST call; selects the device for the calling thread while
 * it runs and restores the previous one).  *ctx receives the context.  Returns CDH_OK,
 * CDH_ERR_INVALID_ARG (ctx NULL, no such device, not an sm_100 device), CDH_ERR_ALLOC, CDH_ERR_CUDA. */
int cdh_create(cdh_ctx **ctx, int device, uint32_t flags);

/*
 * All species-pair histograms of n_frames frames, summed over the frames.
 *
 *  coords          DEVICE pointer, [n_frames][n_total][3] xyz AoS, contiguous, float (precision CDH_F32)
 *                  or double (CDH_F64).
 *                  Coordinates need not be wrapped into the box.  Pairs involving a NaN are dropped.
 *                  Read only during the stream-ordered execution of the call.
 *  n_frames        >= 1.
 *  species_offsets HOST pointer, [n_species + 1]; [0] == 0, non-decreasing, [n_species] == n_total < 2^31;
 *                  the same for every frame.  Empty species are legal (zero histograms).
 *  n_species       1 .. 4096 (the work tables hold one row of segments per species pair and frame).
 *  box_type        CDH_BOX_*.
 *  box             HOST pointer, [n_boxes][9] row-major doubles, ROWS are the box vectors a, b, c
 *                  (the mathematical b of Eq. 5 has them as columns); NULL iff CDH_BOX_NONE.
 *                  CDH_BOX_ORTHO reads the diagonal and requires the off-diagonals to be exactly 0.
 *                  Must be finite and non-singular.
 *  n_boxes         1 (one box for all frames) or n_frames; ignored for CDH_BOX_NONE.
 *  r_max           > 0, finite (CDH_F64: r_max > 1e-100 and n_bins / r_max < 1e100).  Pairs with !(r < (float)r_max) are dropped in every box mode.
 *  n_bins          1 .. 2^22.  Bin width r_max / n_bins; bin = floor(r * (float)(n_bins / r_max)),
 *                  a kept pair whose product rounds up to n_bins goes to bin n_bins - 1.
 *  precision       CDH_F32 or CDH_F64 (constants are then used in double: r_max, n_bins / r_max, the box).
 *  stream          cudaStream_t (as void*), may be 0.  All device work is enqueued on it and `out` is valid once the
 *                  caller has synchronised the stream.  What the HOST does depends on whether the context has seen
 *                  these arguments before (everything but the coords / out pointers and the accumulate flag):
 *                    - first call with a set of arguments: the library builds a PLAN (box constants, work tables,
 *                      kernel variants) and uploads its tables on `stream`.  It allocates the plan's device buffer,
 *                      may grow the context's scratch -- growing a buffer that enqueued work may still read
 *                      synchronises the DEVICE first (cudaDeviceSynchronize) -- and waits for the previous plan's table
 *                      upload before it reuses the pinned staging buffer.  Do not build plans inside a stream capture.
 *                      A call that hits the plan cache MAY be captured into a CUDA graph (cudaStreamBeginCapture ...) and
 *                      replayed any number of times, also between other calls of the context: make the first call with
 *                      these arguments, and synchronise its stream, before the capture begins; a context created with
 *                      CDH_FLAG_TIME_KERNELS records events and cannot be captured.
 *                    - every later call with the same arguments (a trajectory fed frame by frame or chunk by chunk):
 *                      no allocation, no synchronisation, no event wait; it enqueues the repack kernel and the tile
 *                      kernel launch(es) (and one memset of `out` only when `out` is much larger than the coordinates:
 *                      otherwise the repack kernel zeroes it).  The tile kernels are launched with programmatic stream
 *                      serialization: they start while the repack kernel runs and wait on the device before they
 *                      read its output.  The context keeps the 16 most recently used plans.
 *                  If a plan is used on another stream than the one its tables went up on, the call makes that stream
 *                  wait for the upload (cudaStreamWaitEvent).
 *  out             DEVICE pointer, uint64 [n_species*(n_species+1)/2][n_bins], OVERWRITTEN (added to with
 *                  CDH_FLAG_ACCUMULATE).
 *                  Row index of species pair (p <= q): p*n_species - p*(p-1)/2 + (q - p).
 *
 * Host arrays are read during the call only.  Returns CDH_OK or a negative code; every argument check, and every
 * allocation a new plan needs, happens before the first enqueue: on CDH_ERR_INVALID_ARG, CDH_ERR_UNSUPPORTED and
 * CDH_ERR_ALLOC nothing was enqueued and `out` is untouched.
 */
int cdh_histograms(cdh_ctx *ctx, const void *coords, int32_t n_frames,
                   const int32_t *species_offsets, int32_t n_species, int32_t box_type,
                   const double *box, int32_t n_boxes, double r_max, int32_t n_bins,
                   int32_t precision, void *stream, uint64_t *out);

/* Same computation with HOST buffers: `coords` and `out` are host pointers (pageable or pinned).  The
 * library copies the coordinates to the device (one H2D copy), runs cdh_histograms on
 * `stream`, copies the result back (one D2H copy) and SYNCHRONISES the stream before returning.
 * Other arguments, return codes and error behaviour as cdh_histograms. */
int cdh_histograms_host(cdh_ctx *ctx, const void *coords, int32_t n_frames,
                        const int32_t *species_offsets, int32_t n_species, int32_t box_type,
                        const double *box, int32_t n_boxes, double r_max, int32_t n_bins,
                        int32_t precision, void *stream, uint64_t *out);

/*
 * cdh_histograms_host for a trajectory: the frames are processed in chunks of `frames_per_chunk` frames, the
 * H2D copy of chunk c+1 (on a private copy stream, into the other of two chunk buffers) overlapping the kernels of
 * chunk c on `stream`; every frame crosses the bus once and the chunks are summed on the device
 * (Eq. 2; the paper's engine streams frames to the kernels the same way).  Device memory
 * is two chunks instead of the whole trajectory, so the trajectory may be larger than the device memory.
 *
 *  coords            HOST pointer, [n_frames][n_total][3]; page-locked memory is needed for the copies to overlap
 *                    (pageable memory works, the copies then pass through the driver's staging buffer).
 *  frames_per_chunk  >= 1, or 0 = automatic (the fewest frames with 3e10 pairs, at most 1 GiB of coordinates).
 *  box, n_boxes      as cdh_histograms; with n_boxes == n_frames chunk c uses its own frames' boxes.
 *  out               HOST pointer, uint64 [n_hist][n_bins], overwritten.
 * The result is independent of frames_per_chunk (integer sums).  cdh_last_call_info describes the last chunk.
 * Synchronises `stream` before returning.  Other arguments, return codes and error behaviour as cdh_histograms_host.
 */
int cdh_histograms_stream(cdh_ctx *ctx, const void *coords, int32_t n_frames,
                          const int32_t *species_offsets, int32_t n_species, int32_t box_type,
                          const double *box, int32_t n_boxes, double r_max, int32_t n_bins,
                          int32_t precision, int32_t frames_per_chunk, void *stream, uint64_t *out);

/* Destroy the context and free its scratch (synchronises the device).  NULL is accepted. */
int cdh_destroy(cdh_ctx *ctx);

/* Static text for a return code. */
const char *cdh_strerror(int code);

/* Text of the last CUDA error recorded by this context ("" if none); valid until the next call on ctx. */
const char *cdh_last_error(const cdh_ctx *ctx);

/* Introspection of the LAST cdh_histograms call on ctx (host values, no synchronisation):
 *   info[0] = kernels launched by the call      info[1] = work items (tile pairs) scheduled
 *   info[2] = bin-range sweeps                   info[3] = CTAs of the tile kernel
 *   info[4] = threads per CTA                    info[5] = dynamic shared memory bytes per CTA
 *   info[6] = kernel variant id (bit 0 fast path, bit 1 double precision, bit 2 global histogram, bit 3 hybrid (shared window of
 *             the bins + L2 updates for the rest), bits 4-7 box type, bits 8-11 form: ORTHO 0 plain /
 *             1 fused / 2 exact-product rint, TRICLINIC zero structure; bit 12 bin-range split, bit 13 one-CTA-per-SM shape,
 *             bit 14 small-species variant: warps skip below-diagonal and padding-only work; bit 15 no threshold compare in unpadded stages: orthorhombic full-range
 *             private histogram (a slot for every reachable distance, only the first n_bins flushed); bits 16.. j-chunk size)
 *   info[7] = pair slots the tile kernel is scheduled to walk (evaluated pairs incl. masked and padding lanes)
 * Returns CDH_OK or CDH_ERR_INVALID_ARG. */
int cdh_last_call_info(const cdh_ctx *ctx, int64_t info[8]);

/* Device time of a recent cdh_histograms call on a context created with CDH_FLAG_TIME_KERNELS, from CUDA
 * events recorded on the call's stream (a ring of CDH_TIMED_CALLS event sets, one per call):
 *   calls_back = 0 is the last call, 1 the one before, ... (< CDH_TIMED_CALLS and < calls made);
 *   ms[0] = the tile kernel launch(es) (steps S1-S7),
 *   ms[1] = the whole call (table upload of a new plan, zeroing, repack, window sampling, tile kernels).
 * WAITS for that call's last event.  Returns CDH_OK, CDH_ERR_INVALID_ARG (no such flag / no such call /
 * NULL) or CDH_ERR_CUDA. */
#define CDH_TIMED_CALLS 256
int cdh_call_kernel_ms(cdh_ctx *ctx, int calls_back, double ms[2]);

/*
 * Radial distribution function from a summed histogram (Eqs. 1-3):
 *   p_kappa = hist[kappa] / n_frames,   g_kappa = p_kappa / (4 pi (n_pairs / volume) r^2 dr),
 *   dr = r_max / n_bins,  r = (kappa + 1/2) dr  (bin centre).  IEEE double, operations in this order.
 *  hist     DEVICE, uint64 [n_hist][n_bins] (the result of cdh_histograms).
 *  n_pairs  HOST, [n_hist]: unique pairs per frame behind each histogram (N(N-1)/2 or N1*N2); 0 gives inf / NaN rows.
 *  volume   system volume V > 0;  n_frames >= 1: the frames that were summed into hist.
 *  g        DEVICE, double [n_hist][n_bins], overwritten.  Asynchronous on `stream`.
 * Returns CDH_OK, CDH_ERR_INVALID_ARG (nothing enqueued), CDH_ERR_ALLOC or CDH_ERR_CUDA.
 */
int cdh_rdf(cdh_ctx *ctx, const uint64_t *hist, int32_t n_hist, int32_t n_bins, double r_max, int32_t n_frames,
            const double *n_pairs, double volume, void *stream, double *g);

/*
 * The histogram call for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no context, and no cudaMalloc / cudaFree / cudaMallocHost or other allocating
 * CUDA routine on any call.  All device scratch of the call (repacked coordinates, work tables, work counter) lives
 * in ONE static device array of CDH_NOALLOC_SCRATCH_BYTES (1.75 MiB) inside the library, which every GPU holds from
 * the moment it loads the library until the process exits.  Computes what cdh_histograms computes with CDH_F32
 * (same arguments, same integers; Alg. 1, Eq. 4, Eq. 5), overwriting `out`; the kernels are the same tile
 * kernel (no box: the production packed-fp32 variant; periodic boxes: the plain cross-validation variant).
 *
 *  device   CUDA device ordinal (sm_100); coords and out are DEVICE pointers on it, off and box HOST pointers.
 *  stream   cudaStream_t (NULL = default stream); the call is asynchronous on it (it returns once the work tables of
 *           the call have been staged for their host-to-device copy; host arrays may be reused at once).
 * Limits (beyond them the call returns CDH_ERR_UNSUPPORTED, enqueues nothing, and cdh_noalloc_last_error() says
 * which limit): n_frames x (padded particles per frame) <= CDH_NOALLOC_MAX_PADDED_PARTICLES, where every species is
 * padded to a multiple of 4096 particles; n_bins <= CDH_NOALLOC_MAX_BINS; work tables (48 B per frame and species
 * pair + 16 B per i-tile of 1,024 or 4,096 particles + 560 B per box) <= 255.75 KiB.  Larger problems: cdh_histograms.
 * The array is SHARED by all calls on a device and keeps the last call's contents; the call clears what must start
 * at zero.  Calls that overlap on one GPU (two streams, two host threads) race on it: serialise them.  RECORDING into a
 * CUDA graph: a call whose work tables are at most 32,000 bytes (they then travel as a kernel parameter: 3 species x about
 * 100 frames, or a single frame of any size the scratch holds) reads no host memory on the device and can be recorded and
 * replayed, provided the entry point was called once on the device before the capture; with larger tables (copied from
 * host memory of the call) it returns CDH_ERR_UNSUPPORTED on a capturing stream and records nothing.
 * Returns CDH_OK, CDH_ERR_INVALID_ARG, CDH_ERR_UNSUPPORTED or CDH_ERR_CUDA; text via cdh_noalloc_last_error()
 * (per host thread, valid until that thread's next call).
 */
#define CDH_NOALLOC_MAX_PADDED_PARTICLES 131072
#define CDH_NOALLOC_MAX_BINS             32768
#define CDH_NOALLOC_SCRATCH_BYTES        1835008   /* 256 KiB scalars + tables, 1.5 MiB repacked coordinates */
int cdh_histograms_noalloc(int device, const void *coords, int32_t n_frames, const int32_t *species_offsets,
                           int32_t n_species, int32_t box_type, const double *box, int32_t n_boxes,
                           double r_max, int32_t n_bins, void *stream, uint64_t *out);
const char *cdh_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CDH_H */
