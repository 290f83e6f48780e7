// cdh_api.cu -- the C ABI of libcdh (include/cdh.h): context, validation, plans, host dispatch.
//
// A PLAN is everything of a call that depends on its arguments but not on the coordinate values: the box constants,
// the padded layout, the work tables (uploaded once, into the plan's own device buffer), the kernel variants of the
// launch plan with their shared-memory sizes and grids.  Plans are cached per context (cdh_ctx::plans, least recently
// used out), so a trajectory fed frame by frame or chunk by chunk -- the paper's use case, PAPER.md:233, 338 -- pays the
// host work and the table upload once; a call that hits the cache enqueues the repack kernel and the tile
// launches (no memset: the call's scalars are zeroed by the call before it) and touches no allocator and no event.  All device work of a call is enqueued on the caller's stream.
#include <algorithm>
#include <cstdio>
#include <memory>
#include <new>
#include <string>
#include "cdh_host.h"
#include "cdh_math32.cuh"
#include "cdh_f64.cuh"
#include "cdh_rdf.cuh"
#include "cdh_variants.h"

using namespace cdh;

namespace {

struct Launch { Variant v; float lo, hi; };

struct Plan {
    std::vector<unsigned char> key;      // the arguments the plan was built from
    uint64_t stamp = 0;                  // last use (LRU)
    void* d_tables = nullptr;            // segs | rows | boxes | off | pad_off | row_seg | win_lo
    cudaEvent_t uploaded = nullptr;      // the table upload (recorded on up_stream)
    cudaStream_t up_stream = nullptr;
    size_t pk_bytes = 0;                 // repacked coordinates the call needs
    int precision = CDH_F32, box_type = 0, n_hist = 0, n_species = 0, n_frames = 0, n_boxes = 1, n_total = 0;
    uint32_t n_bins = 0, frame_slots = 0, repack_blocks = 0, blocks_per_frame = 0;
    size_t o_rows = 0, o_boxes = 0, o_off = 0, o_pad = 0, o_rowseg = 0, o_win = 0, o_desc = 0;
    bool has_descs = false;
    std::vector<Launch> launches;
    int smem_bytes = 0, mode = MODE_SHARED;
    uint32_t grid = 0, n_items = 0, n_rows = 0, tj = 0, smem_bins = 0, n_stages = 2, keep_bins = 0;
    double r_max = 0.0;
    float rmax_f = 0.f, scale_f = 0.f;
    uint32_t thr2_bits = 0;
    BoxConst64 box0_64;                  // CDH_F64 PBOX variants
    int64_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

}  // namespace

struct cdh_ctx {
    int device = 0;
    uint32_t flags = 0;
    int n_sm = 0;
    int max_smem_optin = 0;
    // device scratch, grown on demand, never shrunk
    void* d_pk = nullptr;        size_t pk_bytes = 0;         // repacked coordinates of the call in flight
    // Four sets of 16 words: [0..2] work counters of the call's tile launches, [4..10] range keys (repack_kernel).  Calls take
    // sets 0 and 1 in turn and the repack kernel of a call zeroes the set of the NEXT one (every kernel of the previous call, the
    // last user of that set, is complete by then: same stream), so a call needs no memset node of its own.
    // A call enqueued while its stream is being CAPTURED into a CUDA graph may be replayed any number of times, between other
    // calls: it uses set 2, zeroed by a memset node of its own, and aims the repack kernel's zeroing at set 3 (a dummy).
    unsigned int* d_scalars = nullptr;
    int scalar_set = 0;
    bool scalars_dirty = false;                               // a call failed half-way: zero both sets before the next one
    void* h_tables = nullptr;    size_t h_tables_bytes = 0;   // pinned staging for a new plan's tables
    cudaEvent_t staged = nullptr;                             // h_tables may be rewritten once this has fired
    bool staged_pending = false;
    void* d_small = nullptr;     size_t small_bytes = 0;      // cdh_rdf: densities
    void* d_io_coords = nullptr; size_t io_coords_bytes = 0;  // cdh_histograms_host staging
    void* d_io_out = nullptr;    size_t io_out_bytes = 0;
    // cdh_histograms_stream: two chunk buffers filled on a private copy stream while the other is being processed
    void* d_chunk[2] = {nullptr, nullptr}; size_t chunk_bytes[2] = {0, 0};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr};
    cudaEvent_t* ev = nullptr;   // CDH_FLAG_TIME_KERNELS: ring of [CDH_TIMED_CALLS][4]: call begin, tile begin, tile end, call end
    uint64_t timed_calls = 0;
    std::vector<std::unique_ptr<Plan>> plans;
    uint64_t stamp = 0;
    std::string err;
    int64_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

namespace {

constexpr size_t kMaxPlans = 16;

struct DeviceGuard {
    int prev = -1; bool ok;
    explicit DeviceGuard(int dev) { ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int cuda_fail(cdh_ctx* c, cudaError_t e, const char* what) {
    c->err = std::string(what) + ": " + cudaGetErrorString(e);
    return CDH_ERR_CUDA;
}
#define CDH_CUDA(call)                                                       \
    do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); } while (0)

// Grows a scratch buffer of the context.  A buffer that enqueued work may still read is not freed under it: the
// device is synchronised first.  Happens only when a call needs more scratch than any call before it.
int grow(cdh_ctx* ctx, void** p, size_t* have, size_t need, bool pinned_host) {
    if (need <= *have) return CDH_OK;
    if (*p) {
        cudaError_t e = cudaDeviceSynchronize();
        if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaDeviceSynchronize");
        if (pinned_host) cudaFreeHost(*p); else cudaFree(*p);
        *p = nullptr; *have = 0;
    }
    const size_t want = need + need / 4 + 4096;
    cudaError_t e = pinned_host ? cudaMallocHost(p, want) : cudaMalloc(p, want);
    if (e != cudaSuccess) { cudaGetLastError(); *p = nullptr; ctx->err = cudaGetErrorString(e); return CDH_ERR_ALLOC; }
    *have = want;
    return CDH_OK;
}

// Pairs one frame evaluates (all species pairs).
double frame_pairs(const int32_t* off, int32_t n_species) {
    double tot = 0.0;
    for (int p = 0; p < n_species; ++p) {
        const double np_ = (double)(off[p + 1] - off[p]);
        tot += 0.5 * np_ * (np_ - 1.0);
        for (int q = p + 1; q < n_species; ++q) tot += np_ * (double)(off[q + 1] - off[q]);
    }
    return tot;
}

#ifndef CDH_SKIP_EFFICIENCY
#define CDH_SKIP_EFFICIENCY 0.95  // the SKIP variants (cdh_sched.cuh) are taken when fewer than this share of the pair slots the
                                  // 1024-particle i-tiles walk are pairs of the problem (measured break-even, one species per
                                  // frame: 16,384 particles, share 0.94: +0.7 %; 24,000 particles, share 0.96: -0.4 %)
#endif
// Small species: the share of the walked pair slots (1024-particle i-tiles: whole stages on the diagonal, padded last tiles)
// that are pairs of the problem decides whether the SKIP variants of the 256-thread kernels pay.
bool small_species(const int32_t* off, int32_t n_species) {
    const double ti256 = 256.0 * kR;
    double walked = 0.0;
    for (int p = 0; p < n_species; ++p) {                       // the count build_tables makes (WorkTables::padded_pairs)
        const double np_ = (double)(off[p + 1] - off[p]), tiles = std::ceil(np_ / ti256);
        walked += ti256 * (tiles * np_ - ti256 * 0.5 * tiles * (tiles - 1.0));          // i-tile t walks j from t * 1024 to n_p
        for (int q = p + 1; q < n_species; ++q) walked += tiles * ti256 * (double)(off[q + 1] - off[q]);
    }
    return walked > 0.0 && frame_pairs(off, n_species) < CDH_SKIP_EFFICIENCY * walked;
}

#ifndef CDH_ITEMS_PER_CTA
#define CDH_ITEMS_PER_CTA 128  // work items per resident CTA the j-chunk size is shrunk for (tail of the dynamic schedule).  Measured
                               // with the item hand-over down to one CTA barrier: 16 / 32 / 64 / 128 / 256 give config 4 1,344 / 1,374 /
                               // 1,385 / 1,388 / 1,385 and config 5 2,191 / 2,191 / 2,191 / 2,201 / 2,203 Gpairs/s (configs 2 and 3 sit at
                               // the smallest j-chunk of a large call, one stage, from 64 on)
#endif
constexpr uint64_t kItemsPerCta = CDH_ITEMS_PER_CTA;
constexpr uint32_t kMinChunk = 32;     // smallest j-chunk (particles)
constexpr uint64_t kDescItems = 262144;  // calls with at most this many work items get the per-item descriptor table (16 MB)
#ifndef CDH_STAGES
#define CDH_STAGES 4           // stages of the TMA ring (cdh_sched.cuh) when the private histogram leaves the room; else 2
#endif

Variant fast_variant(int box_type, int form, int mode, int shape) {
    if (box_type == CDH_BOX_NONE) return fast_variant_none(mode, shape);
    if (box_type == CDH_BOX_ORTHO) return fast_variant_ortho(form, mode, shape);
    return (form & TRI_WIDE) ? fast_variant_tri_wide(form, mode, shape) : fast_variant_tri(form, mode, shape);
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

int smem_fixed(int precision, int n_stages) {
    return precision == CDH_F64 ? tile_smem_fixed<MathF64<BOX_NONE, false>>(n_stages) : tile_smem_fixed<MathFast<BOX_NONE, 0>>(n_stages);
}

}  // namespace

extern "C" const char* cdh_strerror(int code) {
    switch (code) {
        case CDH_OK: return "ok";
        case CDH_ERR_INVALID_ARG: return "invalid argument";
        case CDH_ERR_UNSUPPORTED: return "unsupported";
        case CDH_ERR_ALLOC: return "allocation failed";
        case CDH_ERR_CUDA: return "CUDA runtime error (see cdh_last_error)";
        default: return "unknown error code";
    }
}

extern "C" const char* cdh_last_error(const cdh_ctx* ctx) { return ctx ? ctx->err.c_str() : ""; }

extern "C" int cdh_last_call_info(const cdh_ctx* ctx, int64_t info[8]) {
    if (!ctx || !info) return CDH_ERR_INVALID_ARG;
    for (int k = 0; k < 8; ++k) info[k] = ctx->info[k];
    return CDH_OK;
}

extern "C" int cdh_create(cdh_ctx** out, int device, uint32_t flags) {
    if (!out) return CDH_ERR_INVALID_ARG;
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess) { cudaGetLastError(); return CDH_ERR_CUDA; }
    if (device < 0 || device >= n_dev) return CDH_ERR_INVALID_ARG;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { cudaGetLastError(); return CDH_ERR_CUDA; }
    if (prop.major != 10) return CDH_ERR_INVALID_ARG;            // sm_100a code only
    cdh_ctx* ctx = new (std::nothrow) cdh_ctx;
    if (!ctx) return CDH_ERR_ALLOC;
    ctx->device = device; ctx->flags = flags;
    ctx->n_sm = prop.multiProcessorCount;
    ctx->max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    DeviceGuard g(device);
    if (!g.ok || cudaMalloc(&ctx->d_scalars, 256) != cudaSuccess || cudaMemset(ctx->d_scalars, 0, 256) != cudaSuccess ||
        cudaEventCreateWithFlags(&ctx->staged, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError();
        if (ctx->d_scalars) cudaFree(ctx->d_scalars);
        delete ctx;
        return CDH_ERR_ALLOC;
    }
    if (flags & CDH_FLAG_TIME_KERNELS) {
        ctx->ev = new (std::nothrow) cudaEvent_t[4 * CDH_TIMED_CALLS]();
        if (!ctx->ev) { cdh_destroy(ctx); return CDH_ERR_ALLOC; }
        for (int k = 0; k < 4 * CDH_TIMED_CALLS; ++k)
            if (cudaEventCreate(&ctx->ev[k]) != cudaSuccess) { cudaGetLastError(); cdh_destroy(ctx); return CDH_ERR_ALLOC; }
    }
    *out = ctx;
    return CDH_OK;
}

extern "C" int cdh_call_kernel_ms(cdh_ctx* ctx, int calls_back, double ms[2]) {
    if (!ctx || !ms || !ctx->ev || calls_back < 0 || calls_back >= CDH_TIMED_CALLS ||
        (uint64_t)calls_back >= ctx->timed_calls)
        return CDH_ERR_INVALID_ARG;
    DeviceGuard g(ctx->device);
    const cudaEvent_t* ev = ctx->ev + 4 * ((ctx->timed_calls - 1 - (uint64_t)calls_back) % CDH_TIMED_CALLS);
    float a = 0.f, b = 0.f;
    CDH_CUDA(cudaEventSynchronize(ev[3]));
    CDH_CUDA(cudaEventElapsedTime(&a, ev[1], ev[2]));
    CDH_CUDA(cudaEventElapsedTime(&b, ev[0], ev[3]));
    ms[0] = a; ms[1] = b;
    return CDH_OK;
}

extern "C" int cdh_destroy(cdh_ctx* ctx) {
    if (!ctx) return CDH_OK;
    DeviceGuard g(ctx->device);
    cudaDeviceSynchronize();
    for (auto& p : ctx->plans) { if (p && p->d_tables) cudaFree(p->d_tables); if (p && p->uploaded) cudaEventDestroy(p->uploaded); }
    ctx->plans.clear();
    if (ctx->d_pk) cudaFree(ctx->d_pk);
    if (ctx->d_scalars) cudaFree(ctx->d_scalars);
    if (ctx->d_small) cudaFree(ctx->d_small);
    if (ctx->h_tables) cudaFreeHost(ctx->h_tables);
    if (ctx->d_io_coords) cudaFree(ctx->d_io_coords);
    if (ctx->d_io_out) cudaFree(ctx->d_io_out);
    for (int k = 0; k < 2; ++k) {
        if (ctx->d_chunk[k]) cudaFree(ctx->d_chunk[k]);
        if (ctx->copied[k]) cudaEventDestroy(ctx->copied[k]);
        if (ctx->consumed[k]) cudaEventDestroy(ctx->consumed[k]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->staged) cudaEventDestroy(ctx->staged);
    if (ctx->ev) {
        for (int k = 0; k < 4 * CDH_TIMED_CALLS; ++k) if (ctx->ev[k]) cudaEventDestroy(ctx->ev[k]);
        delete[] ctx->ev;
    }
    cudaGetLastError();
    delete ctx;
    return CDH_OK;
}

static int validate(const void* coords, int32_t n_frames, const int32_t* off, int32_t n_species, int32_t box_type,
                    const double* box, int32_t n_boxes, double r_max, int32_t n_bins, int32_t precision, const void* out) {
    if (!coords || !off || !out) return CDH_ERR_INVALID_ARG;
    if (n_frames < 1 || n_species < 1 || n_species > 4096) return CDH_ERR_INVALID_ARG;
    if (n_bins < 1 || n_bins > (1 << 22)) return CDH_ERR_INVALID_ARG;
    if (!(r_max > 0.0) || !std::isfinite(r_max)) return CDH_ERR_INVALID_ARG;
    if (precision != CDH_F32 && precision != CDH_F64) return CDH_ERR_INVALID_ARG;
    if (box_type != CDH_BOX_NONE && box_type != CDH_BOX_ORTHO && box_type != CDH_BOX_TRICLINIC) return CDH_ERR_INVALID_ARG;
    if (box_type == CDH_BOX_NONE ? (box != nullptr) : (box == nullptr)) return CDH_ERR_INVALID_ARG;
    if (box_type != CDH_BOX_NONE && n_boxes != 1 && n_boxes != n_frames) return CDH_ERR_INVALID_ARG;
    if (off[0] != 0) return CDH_ERR_INVALID_ARG;
    for (int s = 0; s < n_species; ++s) if (off[s + 1] < off[s]) return CDH_ERR_INVALID_ARG;
    if (precision == CDH_F32) {
        if (!((float)r_max > 0.0f) || !std::isfinite((float)r_max)) return CDH_ERR_INVALID_ARG;
        const float scale = (float)((double)n_bins / r_max);
        if (!std::isfinite(scale) || !(scale > 0.0f)) return CDH_ERR_INVALID_ARG;
    } else {
        // the double-precision kernels bin sqrt(d2) < 2^-485 as 0: harmless while it lands in bin 0 and is kept
        if (!(r_max > 1e-100 && (double)n_bins / r_max < 1e100)) return CDH_ERR_INVALID_ARG;
    }
    return CDH_OK;
}

// ---- plans ---------------------------------------------------------------------------------------------------
namespace {

std::vector<unsigned char> plan_key(uint32_t flags, int32_t n_frames, const int32_t* off, int32_t n_species, int32_t box_type,
                                    const double* box, int32_t nb, double r_max, int32_t n_bins, int32_t precision) {
    const int32_t head[7] = {precision, n_frames, n_species, box_type, nb, n_bins, (int32_t)(flags & ~(uint32_t)CDH_FLAG_ACCUMULATE)};
    std::vector<unsigned char> k(sizeof head + sizeof r_max + ((size_t)n_species + 1) * 4 + (size_t)nb * 72);
    unsigned char* w = k.data();
    std::memcpy(w, head, sizeof head); w += sizeof head;
    std::memcpy(w, &r_max, sizeof r_max); w += sizeof r_max;
    std::memcpy(w, off, ((size_t)n_species + 1) * 4); w += ((size_t)n_species + 1) * 4;
    if (nb > 0) std::memcpy(w, box, (size_t)nb * 72);
    return k;
}

#ifndef CDH_GLOBAL_SWEEPS
#define CDH_GLOBAL_SWEEPS 8   // cross-validation kernels only: shared-memory sweeps from which the global-histogram mode takes
                              // over (measured break-even: 200,000 uniform points, 400,000 bins: 8 sweeps 200 vs global 221 Gpairs/s)
#endif
#ifndef CDH_HYBRID_MAX_RATIO
#define CDH_HYBRID_MAX_RATIO 16   // production kernels: n_bins / window above which the shared window is dropped (MODE_GLOBAL):
                                  // it would catch too few pairs to pay for its extra shared update per pair
#endif

// Builds the plan of a call (host work, table upload on `stream`).  Every argument check happens before the first
// enqueue; on error nothing was enqueued.
int build_plan(cdh_ctx* ctx, cudaStream_t stream, int32_t n_frames, const int32_t* off, int32_t n_species, int32_t box_type,
               const double* box, int32_t n_boxes, double r_max, int32_t n_bins, int32_t precision,
               std::vector<unsigned char>&& key, Plan** out_plan) {
    std::unique_ptr<Plan> pl(new (std::nothrow) Plan);
    if (!pl) return CDH_ERR_ALLOC;
    const bool f64 = precision == CDH_F64;
    const int nb = (box_type == CDH_BOX_NONE) ? 0 : n_boxes;
    const size_t n_box_rec = (size_t)(nb > 0 ? nb : 1);

    // ---- host-derived constants ----------------------------------------------------------------
    std::vector<BoxConst> boxes32(f64 ? 0 : n_box_rec);
    std::vector<BoxConst64> boxes64(f64 ? n_box_rec : 0);
    if (f64) std::memset(boxes64.data(), 0, boxes64.size() * sizeof(BoxConst64));
    else std::memset(boxes32.data(), 0, boxes32.size() * sizeof(BoxConst));
    bool prune_all = true, fused_ok = box_type == CDH_BOX_ORTHO;
    for (int b = 0; b < nb; ++b) {
        if (f64) {
            if (!make_box_const64(box_type, box + 9 * (size_t)b, r_max, &boxes64[b])) return CDH_ERR_INVALID_ARG;
            if (ctx->flags & CDH_FLAG_NO_PRUNE) boxes64[b].prune_ok = 0.0;
        } else {
            if (!make_box_const(box_type, box + 9 * (size_t)b, r_max, &boxes32[b])) return CDH_ERR_INVALID_ARG;
            if (boxes32[b].prune_ok == 0.0f) { prune_all = false; fused_ok = false; }
        }
    }
    if (ctx->flags & CDH_FLAG_NO_PRUNE) { prune_all = false; fused_ok = false; }   // tests: 27 shifts everywhere / the plain rint form
    const float rmax_f = (float)r_max;
    const float scale_f = (float)((double)n_bins / r_max);

    // ---- padded layout -------------------------------------------------------------------------
    std::vector<uint32_t> pad_off((size_t)n_species + 1);
    uint64_t slots = 0;
    for (int s = 0; s < n_species; ++s) {
        pad_off[s] = (uint32_t)slots;
        const uint64_t n = (uint64_t)(off[s + 1] - off[s]);
        slots += (n + kPadParticles - 1) / kPadParticles * kPadParticles;
        if (slots > 0x7fffffffull) return CDH_ERR_INVALID_ARG;
    }
    pad_off[n_species] = (uint32_t)slots;
    const uint32_t frame_slots = (uint32_t)slots;
    if ((uint64_t)frame_slots * (uint64_t)n_frames / kGroup > 0xffffffffull) return CDH_ERR_INVALID_ARG;
    const uint32_t blocks_per_frame = (frame_slots + 255) / 256;
    if ((uint64_t)blocks_per_frame * (uint64_t)n_frames > 0x7fffffffull) return CDH_ERR_INVALID_ARG;
    const int n_hist = n_species * (n_species + 1) / 2;

    // ---- where the histogram lives -------------------------------------------------------------
    const bool use_simple_only = !f64 && ((ctx->flags & (CDH_FLAG_SIMPLE_KERNEL | CDH_FLAG_WARP_AGGREGATE | CDH_FLAG_NO_AGGREGATE)) != 0 ||
                                          !(scale_f < 5.0e14f));
    const uint32_t cap_ring = (uint32_t)((ctx->max_smem_optin - smem_fixed(precision, CDH_STAGES)) / 4 - 2);   // bins next to the full ring
    const uint32_t cap_two = (uint32_t)((ctx->max_smem_optin - smem_fixed(precision, 2)) / 4 - 2);              // ... next to two stages
    const uint32_t flag_cap = ctx->flags >> CDH_FLAG_MAX_SMEM_BINS_SHIFT;
    SweepPlan sp; sp.n_sweeps = 1; sp.bins_per_sweep = (uint32_t)n_bins;
    int mode = MODE_SHARED;
    uint32_t smem_bins = (uint32_t)n_bins, n_stages = CDH_STAGES;
    if (ctx->flags & CDH_FLAG_GLOBAL_HIST) { mode = MODE_GLOBAL; smem_bins = 0; }
    else if (flag_cap && flag_cap < (uint32_t)n_bins) {                      // tests: force the bin-range split
        sp = plan_sweeps((uint32_t)n_bins, std::min(flag_cap, cap_two));
        mode = MODE_SPLIT; smem_bins = sp.bins_per_sweep;
    } else if ((uint32_t)n_bins > cap_two) {                                 // wider than a CTA's shared memory
        if (use_simple_only) {
            sp = plan_sweeps((uint32_t)n_bins, cap_two);
            if (sp.n_sweeps >= CDH_GLOBAL_SWEEPS) { sp.n_sweeps = 1; sp.bins_per_sweep = (uint32_t)n_bins; mode = MODE_GLOBAL; smem_bins = 0; }
            else { mode = MODE_SPLIT; smem_bins = sp.bins_per_sweep; }
        } else if ((uint64_t)n_bins > (uint64_t)CDH_HYBRID_MAX_RATIO * cap_two) { mode = MODE_GLOBAL; smem_bins = 0; }
        else { mode = MODE_HYBRID; smem_bins = cap_two; }
    }
    // Orthorhombic box, whole histogram in shared memory: give the private histogram a slot for EVERY reachable distance
    // (wrapped components are within L/2, so d <= |diagonal|/2) and flush only the first n_bins of them.  Stages without
    // padding then need no threshold compare and no trash select (CLEAN form, cdh_fast.cuh).  Exact iff no dropped pair can
    // share a slot with a kept one: bin(thr2) >= n_bins, and no kept pair rounds up into slot n_bins (reading Q3).
    uint32_t keep_bins = 0;
#ifndef CDH_ORTHO_CLEAN
#define CDH_ORTHO_CLEAN 1
#endif
    if (CDH_ORTHO_CLEAN && box_type == CDH_BOX_ORTHO && mode == MODE_SHARED && !use_simple_only && !(ctx->flags & CDH_FLAG_NO_PRUNE)) {
        // the two bins that decide it, by the pinned operations of the precision: of the first dropped distance and of the last kept one
        double b_thr, b_prev;
        if (f64) {
            const double scale_d = (double)n_bins / r_max;
            b_thr = std::floor(r_max * scale_d); b_prev = std::floor(std::nextafter(r_max, 0.0) * scale_d);
        } else {
            const float thr2 = bits_f32(d2_threshold_bits(rmax_f));
            b_thr = (double)floorf(sqrtf(thr2) * scale_f); b_prev = (double)floorf(sqrtf(std::nextafterf(thr2, 0.0f)) * scale_f);
        }
        double d2max = 0.0;
        for (int b = 0; b < nb; ++b) {
            double acc = 0.0;
            for (int c = 0; c < 3; ++c) {
                const double h = std::fabs(f64 ? boxes64[b].L[c] : (double)boxes32[b].L[c]) * (0.5 + std::ldexp(1.0, -18));
                acc += h * h;
            }
            d2max = std::fmax(d2max, acc);
        }
        const double slots = std::floor(std::sqrt(d2max) * (f64 ? (double)n_bins / r_max : (double)scale_f) * (1.0 + 1e-6)) + 3.0;
        if (b_thr >= (double)n_bins && b_prev <= (double)(n_bins - 1) && slots < 4.0e6 && slots > (double)n_bins) {
            const uint32_t all = (uint32_t)slots;
            // measured: config 4 (3 resident CTAs either way) 1,258 -> 1,356 Gpairs/s; config 2 (2 instead of 3 resident CTAs)
            // 1,231 -> 1,308: the two instructions saved per pair outweigh the lost CTA, so the form is taken whenever it fits
            if (all <= cap_two) { keep_bins = (uint32_t)n_bins; smem_bins = all; }
        }
    }
    // Triclinic box: the zero-shift candidates reach several r_max, so a slot for every distance does not fit; instead the
    // CLEAN stages clamp d2 to the threshold (one FMNMX for compare + select, bin_fast2 CLAMP): every dropped pair lands in the
    // slot of bin(thr2), which must be one of the two spare slots (n_bins, n_bins + 1) and is then not flushed -- so no kept
    // pair may round up into slot n_bins (reading Q3).  Same two decisive bins as above.
    if (CDH_ORTHO_CLEAN && !f64 && box_type == CDH_BOX_TRICLINIC && mode == MODE_SHARED && !use_simple_only) {
        const uint32_t tb = d2_threshold_bits(rmax_f);
        if (tb < 0x7f800000u) {
            const float thr2 = bits_f32(tb);
            const float b_thr = floorf(sqrtf(thr2) * scale_f), b_prev = floorf(sqrtf(std::nextafterf(thr2, 0.0f)) * scale_f);
            if ((b_thr == (float)n_bins || b_thr == (float)n_bins + 1.0f) && b_prev <= (float)(n_bins - 1)) keep_bins = (uint32_t)n_bins;
        }
    }
    if (mode != MODE_GLOBAL && smem_bins > cap_ring) n_stages = 2;
    if (n_stages > 2 && mode != MODE_GLOBAL) {
        // two stages instead of four where that lets one more 256-thread CTA fit an SM (config 2's full-range histogram:
        // 76 KB instead of 82 KB per CTA, 3 instead of 2 CTAs); the depth of the ring itself is worth nothing measurable
        const int reg_ctas = (f64 || box_type == CDH_BOX_TRICLINIC || use_simple_only) ? 2 : 3;   // what the kernels' registers allow
        const int per_sm = 228 * 1024;
        const int b4 = smem_fixed(precision, (int)n_stages) + 4 * ((int)smem_bins + 2) + 1024, b2 = smem_fixed(precision, 2) + 4 * ((int)smem_bins + 2) + 1024;
        if (std::min(reg_ctas, per_sm / b2) > std::min(reg_ctas, per_sm / b4)) n_stages = 2;
    }
    const int smem_bytes = smem_fixed(precision, (int)n_stages) + 4 * ((int)smem_bins + 2);
#ifndef CDH_BIG_BELOW_CTAS_NONE
#define CDH_BIG_BELOW_CTAS_NONE 3
#endif
#ifndef CDH_BIG_BELOW_CTAS
#define CDH_BIG_BELOW_CTAS 2     // the one-CTA-per-SM shape is taken when fewer than this many 256-thread CTAs fit one SM (measured with 3:
                                 // config 2 1,309 -> 1,170, config 3 784 -> 694 Gpairs/s: the 1,024-thread shape is bounded to 64 registers)
#endif
    // no box: the 1,024-thread kernel needs 62 registers and loses nothing to the cap of 64, so it is also taken where only two
    // 256-thread CTAs (16 warps per SM instead of 32) would fit (measured, 25,000 bins: 2,040 -> 2,111 Gpairs/s)
    const int big_below = (box_type == CDH_BOX_NONE && !f64 && !use_simple_only) ? CDH_BIG_BELOW_CTAS_NONE : CDH_BIG_BELOW_CTAS;
    const bool big = big_below * (smem_bytes + 1024) > 228 * 1024 || mode == MODE_HYBRID;          // one CTA per SM
    // the SKIP kernels also carry the late claim of work items (cdh_sched.cuh), which pays where a CTA gets only a few items:
    // they are taken as well when the call has fewer than about 6 one-stage items per resident CTA (measured, single frames,
    // calls back to back: 20,000 points no box 1,267 -> 1,412, orthorhombic 851 -> 1,044; 30,000 points triclinic 710 -> 761;
    // 40,000 points, 7 items per CTA: -0.6 / -2.5 / +1.3 %, left alone)
    const bool few_items = frame_pairs(off, n_species) * (double)n_frames < 6.0 * 3.0 * (double)ctx->n_sm * 1024.0 * (double)kStageParticles;
    const bool skip = !big && mode == MODE_SHARED && !use_simple_only && (small_species(off, n_species) || few_items);
    const int shape = big ? SHAPE_BIG : (skip ? SHAPE_256_SKIP : SHAPE_256);

    // ---- launch plan ----------------------------------------------------------------------------
    // Every tile launch of the call owns an interval (lo, hi] of the fractional-coordinate range the repack kernel
    // measures, and exactly one of them does the work (cdh_math32.cuh launch_begin).
    //   ORTHO: fused rint up to 1.49 (exact-product form if the host found no fused constants for some box),
    //          magic-number rint up to 2^20, library rintf beyond;  TRICLINIC: fast path up to 1.49 (n in {-1,0,1}),
    //          wide fast path up to 64, definition beyond.
    const float kInf = INFINITY, kSmall = 1.49f, kWide = 64.0f, kMagic = 1048576.0f;
    int form = 0;
    bool pbox = false;
    if (f64) {
        pbox = box_type == CDH_BOX_TRICLINIC && nb == 1;      // one box: constants through the parameter bank
        pl->launches.push_back({f64_variant(box_type, pbox, mode, shape), -kInf, kInf});
    } else {
        const int simple_mode = (mode == MODE_SHARED || mode == MODE_SPLIT) ? MODE_SPLIT : MODE_GLOBAL;
        const int var = (ctx->flags & CDH_FLAG_WARP_AGGREGATE) ? VAR_SIMPLE_MATCH : (ctx->flags & CDH_FLAG_NO_AGGREGATE) ? VAR_SIMPLE_PLAIN : VAR_SIMPLE;
        const Variant vs = simple_variant(box_type, var, simple_mode, big ? SHAPE_BIG : SHAPE_256);
        auto fast_of = [&](int f) { return fast_variant(box_type, f, mode, shape); };
        if (use_simple_only) pl->launches.push_back({vs, -kInf, kInf});
        else if (box_type == CDH_BOX_NONE) pl->launches.push_back({fast_of(0), -kInf, kInf});
        else if (box_type == CDH_BOX_ORTHO) {
            const bool plain_only = (ctx->flags & CDH_FLAG_NO_PRUNE) != 0;     // tests: the pinned 5-operation form everywhere
            form = plain_only ? ORTHO_PLAIN : fused_ok ? ORTHO_FUSED : ORTHO_EXACT;
            if (plain_only) pl->launches.push_back({fast_of(ORTHO_PLAIN), -kInf, kMagic});
            else { pl->launches.push_back({fast_of(form), -kInf, kSmall}); pl->launches.push_back({fast_of(ORTHO_PLAIN), kSmall, kMagic}); }
            pl->launches.push_back({vs, kMagic, kInf});
        } else {
            // all boxes prunable: the zero structure shared by B and B^-1 picks the form; else the 27-shift search for every pair
            form = prune_all ? tri_kind(boxes32.data(), nb) : (TRI_GENERAL | TRI_NOPRUNE);
            pl->launches.push_back({fast_of(form), -kInf, kSmall});
            pl->launches.push_back({fast_of(form | TRI_WIDE), kSmall, kWide});      // unwrapped coordinates, up to 64 cells
            pl->launches.push_back({vs, kWide, kInf});
        }
    }
    for (const Launch& l : pl->launches) if (!l.v.fn) { ctx->err = "kernel variant not built"; return CDH_ERR_UNSUPPORTED; }
    const Variant vf = pl->launches[0].v;
    const uint32_t ti = (uint32_t)vf.threads * kR;

    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");
    for (const Launch& l : pl->launches)
        CDH_CUDA(cudaFuncSetAttribute(l.v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    int resident = 0;      // CTAs of the production variant that fit one SM (registers, shared memory)
    CDH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, vf.fn, vf.threads, (size_t)smem_bytes));
    if (resident < 1) resident = 1;
    const uint32_t grid_full = (uint32_t)ctx->n_sm * (uint32_t)resident;

    WorkTables wt;
    uint32_t tj = 8192;
    for (;; tj >>= 1) {
        build_tables(n_frames, off, n_species, nb > 0 ? nb : 1, (uint32_t)n_bins, sp, ti, tj, pad_off, frame_slots, &wt);
        if (wt.n_items >= kItemsPerCta * grid_full) break;
        // small calls: j-chunks below one stage (the stage is then partly used) until every resident CTA has an item --
        // a 2,000-particle frame becomes 94 items of 1024 x 32 pairs instead of 12 of 1024 x 256 (launch-latency regime)
        if (tj <= (uint32_t)kStageParticles && (wt.n_items >= grid_full || tj == kMinChunk)) break;
    }
    if (wt.n_items >= 0xf0000000ull || wt.rows.size() >= 0x7fffffffull) return CDH_ERR_INVALID_ARG;
    std::vector<int32_t> row_seg((size_t)n_hist, -1);          // first segment of each histogram row (window_kernel)
    for (size_t k = wt.segs.size(); k-- > 0;) row_seg[wt.segs[k].hist] = (int32_t)k;

    // ---- tables: staged in pinned memory, uploaded once into the plan's own device buffer --------------------------
    const size_t box_rec = f64 ? sizeof(BoxConst64) : sizeof(BoxConst);
    const size_t b_segs = align256(wt.segs.size() * sizeof(Seg) + 1), b_rows = align256(wt.rows.size() * sizeof(Row)),
                 b_boxes = align256(n_box_rec * box_rec), b_off = align256(((size_t)n_species + 1) * 4),
                 b_rowseg = align256((size_t)n_hist * 4);
    pl->o_rows = b_segs; pl->o_boxes = pl->o_rows + b_rows; pl->o_off = pl->o_boxes + b_boxes; pl->o_pad = pl->o_off + b_off;
    pl->o_rowseg = pl->o_pad + b_off; pl->o_win = pl->o_rowseg + b_rowseg;
    // one descriptor per item, fetched by the kernel one item ahead (cdh_sched.cuh); calls with very many items do without
    pl->has_descs = wt.n_items > 0 && wt.n_items <= kDescItems && !(ctx->flags & CDH_FLAG_NO_ITEM_TABLE);
    pl->o_desc = pl->o_win + b_rowseg;
    const size_t tables = pl->o_desc + (pl->has_descs ? align256((size_t)wt.n_items * sizeof(ItemDesc)) : 0);
    int rc;
    if (ctx->staged_pending) { CDH_CUDA(cudaEventSynchronize(ctx->staged)); ctx->staged_pending = false; }
    if ((rc = grow(ctx, &ctx->h_tables, &ctx->h_tables_bytes, tables, true)) != CDH_OK) return rc;
    const size_t pk_need = (size_t)n_frames * frame_slots * 3 * (f64 ? sizeof(double) : sizeof(float));
    if ((rc = grow(ctx, &ctx->d_pk, &ctx->pk_bytes, pk_need > 0 ? pk_need : 16, false)) != CDH_OK) return rc;
    if (cudaMalloc(&pl->d_tables, tables) != cudaSuccess) { cudaGetLastError(); pl->d_tables = nullptr; ctx->err = "plan tables"; return CDH_ERR_ALLOC; }
    char* h = (char*)ctx->h_tables;
    std::memset(h, 0, tables);
    std::memcpy(h, wt.segs.data(), wt.segs.size() * sizeof(Seg));
    std::memcpy(h + pl->o_rows, wt.rows.data(), wt.rows.size() * sizeof(Row));
    std::memcpy(h + pl->o_boxes, f64 ? (const void*)boxes64.data() : (const void*)boxes32.data(), n_box_rec * box_rec);
    std::memcpy(h + pl->o_off, off, ((size_t)n_species + 1) * 4);
    std::memcpy(h + pl->o_pad, pad_off.data(), ((size_t)n_species + 1) * 4);
    std::memcpy(h + pl->o_rowseg, row_seg.data(), (size_t)n_hist * 4);
    if (pl->has_descs) {
        ItemDesc* dd = reinterpret_cast<ItemDesc*>(h + pl->o_desc);
        for (size_t r = 0; r + 1 < wt.rows.size(); ++r)
            for (uint32_t it = wt.rows[r].item_prefix; it < wt.rows[r + 1].item_prefix; ++it) {
                dd[it].seg = wt.segs[wt.rows[r].seg];
                dd[it].i0 = wt.rows[r].i0; dd[it].jc = wt.rows[r].jc0 + (it - wt.rows[r].item_prefix); dd[it].pad_[0] = it;
            }
    }
    cudaError_t e = cudaEventCreateWithFlags(&pl->uploaded, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMemcpyAsync(pl->d_tables, h, tables, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->staged, stream);
    if (e == cudaSuccess) e = cudaEventRecord(pl->uploaded, stream);
    if (e != cudaSuccess) {
        cudaFree(pl->d_tables); pl->d_tables = nullptr;
        if (pl->uploaded) cudaEventDestroy(pl->uploaded);
        return cuda_fail(ctx, e, "plan table upload");
    }
    ctx->staged_pending = true;
    pl->up_stream = stream;

    pl->key = std::move(key);
    pl->pk_bytes = pk_need;
    pl->precision = precision; pl->box_type = box_type; pl->n_hist = n_hist; pl->n_species = n_species; pl->n_frames = n_frames;
    pl->n_boxes = nb > 0 ? nb : 1; pl->n_total = off[n_species];
    pl->n_bins = (uint32_t)n_bins; pl->frame_slots = frame_slots; pl->blocks_per_frame = blocks_per_frame;
    pl->repack_blocks = blocks_per_frame * (uint32_t)n_frames;
    pl->smem_bytes = smem_bytes; pl->mode = mode; pl->n_items = (uint32_t)wt.n_items; pl->n_rows = (uint32_t)wt.rows.size() - 1;
    pl->grid = grid_full < pl->n_items ? grid_full : pl->n_items;
    pl->tj = tj; pl->smem_bins = smem_bins; pl->n_stages = n_stages; pl->keep_bins = keep_bins;
    pl->r_max = r_max; pl->rmax_f = rmax_f; pl->scale_f = scale_f; pl->thr2_bits = f64 ? 0u : d2_threshold_bits(rmax_f);
    if (f64) pl->box0_64 = boxes64[0];
    const int n_launch = (frame_slots > 0 ? 1 : 0) + (wt.n_items > 0 ? (int)pl->launches.size() + (mode == MODE_HYBRID ? 1 : 0) : 0);
    pl->info[0] = n_launch; pl->info[1] = (int64_t)wt.n_items; pl->info[2] = sp.n_sweeps; pl->info[3] = pl->grid;
    pl->info[4] = vf.threads; pl->info[5] = smem_bytes;
    pl->info[6] = (f64 ? 2 : (use_simple_only ? 0 : 1)) | ((int)(mode == MODE_GLOBAL) << 2) | ((int)(mode == MODE_HYBRID) << 3) | (box_type << 4) |
                  ((form & 15) << 8) | ((int)(mode == MODE_SPLIT) << 12) | ((int)big << 13) | ((int)skip << 14) | ((int)(keep_bins != 0) << 15) | ((int64_t)tj << 16);
    pl->info[7] = (int64_t)wt.padded_pairs;

    // least recently used plan out (its tables may still be read by enqueued work: wait for the device first)
    if (ctx->plans.size() >= kMaxPlans) {
        size_t victim = 0;
        for (size_t k = 1; k < ctx->plans.size(); ++k) if (ctx->plans[k]->stamp < ctx->plans[victim]->stamp) victim = k;
        cudaDeviceSynchronize();
        if (ctx->plans[victim]->d_tables) cudaFree(ctx->plans[victim]->d_tables);
        if (ctx->plans[victim]->uploaded) cudaEventDestroy(ctx->plans[victim]->uploaded);
        ctx->plans.erase(ctx->plans.begin() + (long)victim);
    }
    *out_plan = pl.get();
    ctx->plans.push_back(std::move(pl));
    return CDH_OK;
}

// Enqueues the call on `stream`: zeroing, repack, (window), tile launch(es).
int enqueue_plan(cdh_ctx* ctx, const Plan& pl, const void* coords, cudaStream_t stream, uint64_t* out) {
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");
    const bool f64 = pl.precision == CDH_F64;
    char* d = (char*)pl.d_tables;
    const bool timing = ctx->ev != nullptr;
    cudaEvent_t* ev = timing ? ctx->ev + 4 * (ctx->timed_calls % CDH_TIMED_CALLS) : nullptr;
    cudaStreamCaptureStatus cap_status = cudaStreamCaptureStatusNone;
    CDH_CUDA(cudaStreamIsCapturing(stream, &cap_status));
    const bool capturing = cap_status == cudaStreamCaptureStatusActive;   // the call is being recorded into a CUDA graph
    // the tables went up on another stream (under capture the caller has seen to it: include/cdh.h)
    if (stream != pl.up_stream && !capturing) CDH_CUDA(cudaStreamWaitEvent(stream, pl.uploaded, 0));
    if (timing) CDH_CUDA(cudaEventRecord(ev[0], stream));
    unsigned int* scalars; unsigned int* scalars_next;
    if (capturing) {
        scalars = ctx->d_scalars + 32; scalars_next = ctx->d_scalars + 48;
        CDH_CUDA(cudaMemsetAsync(scalars, 0, 64, stream));       // a node of the graph: every replay starts from zero
    } else {
        if (ctx->scalars_dirty) { CDH_CUDA(cudaMemsetAsync(ctx->d_scalars, 0, 128, stream)); ctx->scalar_set = 0; }
        ctx->scalars_dirty = true;                               // until this call is enqueued completely
        scalars = ctx->d_scalars + 16 * ctx->scalar_set; scalars_next = ctx->d_scalars + 16 * (ctx->scalar_set ^ 1);
    }
    const bool zero_out = !(ctx->flags & CDH_FLAG_ACCUMULATE);
    const uint64_t out_count = (uint64_t)pl.n_hist * (uint64_t)pl.n_bins;
    // the repack kernel zeroes the result on its way unless that would be most of its work (few particles, very many bins)
    const bool fold_zero = zero_out && pl.frame_slots > 0 && out_count <= 64ull * 256ull * pl.repack_blocks;
    if (zero_out && !fold_zero) CDH_CUDA(cudaMemsetAsync(out, 0, out_count * sizeof(uint64_t), stream));

    // ---- K0 repack -----------------------------------------------------------------------------
    if (pl.frame_slots > 0) {
        if (f64) {
            RepackParams64 rp;
            rp.coords = (const double*)coords; rp.pk = (double*)ctx->d_pk;
            rp.off = (const int32_t*)(d + pl.o_off); rp.pad_off = (const uint32_t*)(d + pl.o_pad);
            rp.range_keys = scalars + 4; rp.reset = scalars_next; rp.boxes = (const BoxConst64*)(d + pl.o_boxes);
            rp.n_species = pl.n_species; rp.n_total = pl.n_total; rp.n_frames = pl.n_frames;
            rp.box_type = pl.box_type; rp.n_boxes = pl.n_boxes;
            rp.frame_slots = pl.frame_slots; rp.blocks_per_frame = pl.blocks_per_frame;
            rp.zero = fold_zero ? (unsigned long long*)out : nullptr; rp.zero_count = out_count;
            repack_kernel_f64<<<pl.repack_blocks, 256, 0, stream>>>(rp);
        } else {
            RepackParams rp;
            rp.coords = (const float*)coords; rp.pk = (float*)ctx->d_pk;
            rp.off = (const int32_t*)(d + pl.o_off); rp.pad_off = (const uint32_t*)(d + pl.o_pad);
            rp.range_keys = scalars + 4; rp.reset = scalars_next; rp.boxes = (const BoxConst*)(d + pl.o_boxes);
            rp.n_species = pl.n_species; rp.n_total = pl.n_total; rp.n_frames = pl.n_frames;
            rp.box_type = pl.box_type; rp.n_boxes = pl.n_boxes;
            rp.frame_slots = pl.frame_slots; rp.blocks_per_frame = pl.blocks_per_frame;
            rp.zero = fold_zero ? (unsigned long long*)out : nullptr; rp.zero_count = out_count;
            repack_kernel<<<pl.repack_blocks, 256, 0, stream>>>(rp);
        }
        CDH_CUDA(cudaGetLastError());
    }

    // ---- K1 tile kernel(s) ---------------------------------------------------------------------
    if (timing) CDH_CUDA(cudaEventRecord(ev[1], stream));
    if (pl.n_items > 0) {
        TileParams tp; TileParams64 tp64;
        TileCommon& c = f64 ? static_cast<TileCommon&>(tp64) : static_cast<TileCommon&>(tp);
        c.segs = (const Seg*)d; c.rows = (const Row*)(d + pl.o_rows);
        c.descs = pl.has_descs ? (const ItemDesc*)(d + pl.o_desc) : nullptr;
        c.out = (unsigned long long*)out; c.range_keys = scalars + 4; c.win_lo = (const uint32_t*)(d + pl.o_win);
        c.n_rows = pl.n_rows; c.n_items = pl.n_items; c.n_bins = pl.n_bins; c.tj = pl.tj; c.smem_bins = pl.smem_bins;
        c.n_stages = pl.n_stages; c.claim_ahead = (uint64_t)pl.n_items >= 16ull * pl.grid ? 1u : 0u;
        if (f64) {
            tp64.pk = (const double*)ctx->d_pk; tp64.boxes = (const BoxConst64*)(d + pl.o_boxes);
            tp64.rmax = pl.r_max; tp64.scale = (double)pl.n_bins / pl.r_max; tp64.box0 = pl.box0_64; tp64.keep_bins = pl.keep_bins;
        } else {
            tp.pk = (const float*)ctx->d_pk; tp.boxes = (const BoxConst*)(d + pl.o_boxes);
            tp.rmax = pl.rmax_f; tp.scale = pl.scale_f; tp.thr2_bits = pl.thr2_bits; tp.one = 1.0f; tp.one_u = 1.0f;
        }
        if (pl.mode == MODE_HYBRID) {       // K0b: the shared-memory window of every histogram row
            if (f64) {
                WindowParams<double, BoxConst64> wp;
                wp.pk = tp64.pk; wp.segs = c.segs; wp.row_seg = (const int32_t*)(d + pl.o_rowseg); wp.boxes = tp64.boxes;
                wp.win_lo = (uint32_t*)(d + pl.o_win); wp.box_type = pl.box_type; wp.n_bins = pl.n_bins; wp.window = pl.smem_bins;
                wp.scale = (float)((double)pl.n_bins / pl.r_max);
                window_kernel<double, BoxConst64><<<pl.n_hist, 256, 0, stream>>>(wp);
            } else {
                WindowParams<float, BoxConst> wp;
                wp.pk = tp.pk; wp.segs = c.segs; wp.row_seg = (const int32_t*)(d + pl.o_rowseg); wp.boxes = tp.boxes;
                wp.win_lo = (uint32_t*)(d + pl.o_win); wp.box_type = pl.box_type; wp.n_bins = pl.n_bins; wp.window = pl.smem_bins;
                wp.scale = pl.scale_f;
                window_kernel<float, BoxConst><<<pl.n_hist, 256, 0, stream>>>(wp);
            }
            CDH_CUDA(cudaGetLastError());
        }
        for (size_t k = 0; k < pl.launches.size(); ++k) {
            c.counter = scalars + k;
            // the orthorhombic full-range form belongs to the first launch (fractional range <= 1.49); the triclinic clamp to both fast ones
            if (!f64) { tp.range_lo = pl.launches[k].lo; tp.range_hi = pl.launches[k].hi; tp.keep_bins = (k == 0 || (pl.box_type == CDH_BOX_TRICLINIC && k == 1)) ? pl.keep_bins : 0u; }
            void* args[1] = {f64 ? (void*)&tp64 : (void*)&tp};
            // programmatic stream serialization: the launch may begin while the kernel before it (repack, window or the
            // previous tile launch) still runs; the kernel waits (griddepcontrol.wait) before it reads what they wrote
            cudaLaunchAttribute attr[1];
            attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            attr[0].val.programmaticStreamSerializationAllowed = 1;
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(pl.grid); cfg.blockDim = dim3((unsigned)pl.launches[k].v.threads);
            cfg.dynamicSmemBytes = (size_t)pl.smem_bytes; cfg.stream = stream;
            cfg.attrs = attr; cfg.numAttrs = (ctx->flags & CDH_FLAG_NO_PDL) ? 0 : 1;
            CDH_CUDA(cudaLaunchKernelExC(&cfg, pl.launches[k].v.fn, args));
        }
    }
    if (timing) {
        CDH_CUDA(cudaEventRecord(ev[2], stream));
        CDH_CUDA(cudaEventRecord(ev[3], stream));
        ++ctx->timed_calls;
    }
    for (int k = 0; k < 8; ++k) ctx->info[k] = pl.info[k];
    if (!capturing) {
        if (pl.frame_slots > 0) ctx->scalar_set ^= 1;            // the repack kernel has zeroed the other set
        ctx->scalars_dirty = false;
    }
    return CDH_OK;
}

}  // namespace

extern "C" int cdh_histograms(cdh_ctx* ctx, const void* coords, int32_t n_frames, const int32_t* off,
                              int32_t n_species, int32_t box_type, const double* box, int32_t n_boxes,
                              double r_max, int32_t n_bins, int32_t precision, void* stream_, uint64_t* out) {
    if (!ctx) return CDH_ERR_INVALID_ARG;
    int rc = validate(coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, precision, out);
    if (rc != CDH_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    ctx->err.clear();
    const int nb = (box_type == CDH_BOX_NONE) ? 0 : n_boxes;
    std::vector<unsigned char> key = plan_key(ctx->flags, n_frames, off, n_species, box_type, box, nb, r_max, n_bins, precision);
    Plan* pl = nullptr;
    for (auto& p : ctx->plans)
        if (p->key.size() == key.size() && std::memcmp(p->key.data(), key.data(), key.size()) == 0) { pl = p.get(); break; }
    if (!pl) {
        rc = build_plan(ctx, stream, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, precision, std::move(key), &pl);
        if (rc != CDH_OK) return rc;
    }
    pl->stamp = ++ctx->stamp;
    return enqueue_plan(ctx, *pl, coords, stream, out);
}

extern "C" int cdh_histograms_host(cdh_ctx* ctx, const void* coords, int32_t n_frames, const int32_t* off,
                                   int32_t n_species, int32_t box_type, const double* box, int32_t n_boxes,
                                   double r_max, int32_t n_bins, int32_t precision, void* stream_, uint64_t* out) {
    if (!ctx) return CDH_ERR_INVALID_ARG;
    int rc = validate(coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, precision, out);
    if (rc != CDH_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");
    const size_t cbytes = (size_t)n_frames * (size_t)off[n_species] * 3 * (precision == CDH_F64 ? sizeof(double) : sizeof(float));
    const size_t obytes = (size_t)(n_species * (n_species + 1) / 2) * (size_t)n_bins * sizeof(uint64_t);
    if ((rc = grow(ctx, &ctx->d_io_coords, &ctx->io_coords_bytes, cbytes > 0 ? cbytes : 16, false)) != CDH_OK) return rc;
    if ((rc = grow(ctx, &ctx->d_io_out, &ctx->io_out_bytes, obytes, false)) != CDH_OK) return rc;
    if (cbytes) CDH_CUDA(cudaMemcpyAsync(ctx->d_io_coords, coords, cbytes, cudaMemcpyHostToDevice, stream));   // one H2D copy
    const uint32_t saved_flags = ctx->flags;
    ctx->flags &= ~CDH_FLAG_ACCUMULATE;                       // the device result of this entry point is scratch: overwrite
    rc = cdh_histograms(ctx, ctx->d_io_coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins,
                        precision, stream_, (uint64_t*)ctx->d_io_out);
    ctx->flags = saved_flags;
    if (rc != CDH_OK) return rc;
    CDH_CUDA(cudaMemcpyAsync(out, ctx->d_io_out, obytes, cudaMemcpyDeviceToHost, stream));                      // one D2H copy
    CDH_CUDA(cudaStreamSynchronize(stream));
    return CDH_OK;
}

#ifndef CDH_STREAM_CHUNK_PAIRS
#define CDH_STREAM_CHUNK_PAIRS 3.0e10   // automatic chunk: the fewest frames with this many pairs (about 25 ms of tile kernel: the
                                        // 0.1 ms a chunk costs -- tables, zeroing, the tail of its wave -- stays below 0.5 %;
                                        // measured on config 4: 7-frame chunks of 6 ms were 1.3 % slower than one call)
#endif
#ifndef CDH_STREAM_CHUNK_BYTES
#define CDH_STREAM_CHUNK_BYTES (1ull << 30)  // and at most this many coordinate bytes per chunk buffer
#endif

extern "C" int cdh_histograms_stream(cdh_ctx* ctx, const void* coords, int32_t n_frames, const int32_t* off,
                                     int32_t n_species, int32_t box_type, const double* box, int32_t n_boxes,
                                     double r_max, int32_t n_bins, int32_t precision, int32_t frames_per_chunk,
                                     void* stream_, uint64_t* out) {
    if (!ctx || frames_per_chunk < 0) return CDH_ERR_INVALID_ARG;
    int rc = validate(coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, precision, out);
    if (rc != CDH_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");
    const size_t fbytes = (size_t)off[n_species] * 3 * (precision == CDH_F64 ? sizeof(double) : sizeof(float));
    const size_t obytes = (size_t)(n_species * (n_species + 1) / 2) * (size_t)n_bins * sizeof(uint64_t);
    int64_t fpc = frames_per_chunk;
    if (fpc == 0) {
        const double pairs = frame_pairs(off, n_species);
        fpc = pairs > 0.0 ? (int64_t)std::ceil(CDH_STREAM_CHUNK_PAIRS / pairs) : n_frames;
        if (fbytes > 0 && (uint64_t)fpc * fbytes > CDH_STREAM_CHUNK_BYTES) fpc = (int64_t)(CDH_STREAM_CHUNK_BYTES / fbytes);
    }
    if (fpc < 1) fpc = 1;
    if (fpc > n_frames) fpc = n_frames;
    if (!ctx->copy_stream) {
        CDH_CUDA(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            CDH_CUDA(cudaEventCreateWithFlags(&ctx->copied[k], cudaEventDisableTiming));
            CDH_CUDA(cudaEventCreateWithFlags(&ctx->consumed[k], cudaEventDisableTiming));
        }
    }
    const size_t chunk_bytes = (size_t)fpc * fbytes;
    const int64_t n_chunks = ((int64_t)n_frames + fpc - 1) / fpc;
    for (int k = 0; k < (n_chunks > 1 ? 2 : 1); ++k)
        if ((rc = grow(ctx, &ctx->d_chunk[k], &ctx->chunk_bytes[k], chunk_bytes > 0 ? chunk_bytes : 16, false)) != CDH_OK) return rc;
    if ((rc = grow(ctx, &ctx->d_io_out, &ctx->io_out_bytes, obytes, false)) != CDH_OK) return rc;
    // the buffers may still be read by work a caller enqueued on `stream` before this call (an earlier call of this entry
    // point ends synchronised, so in practice this orders nothing): the first copies wait for the stream's present tail
    CDH_CUDA(cudaEventRecord(ctx->consumed[0], stream));
    CDH_CUDA(cudaEventRecord(ctx->consumed[1], stream));
    const uint32_t saved_flags = ctx->flags;
    for (int64_t c = 0; c < n_chunks && rc == CDH_OK; ++c) {
        const int k = (int)(c & 1);
        const int64_t f0 = c * fpc;
        const int32_t nf = (int32_t)((int64_t)n_frames - f0 < fpc ? (int64_t)n_frames - f0 : fpc);
        cudaError_t e = cudaStreamWaitEvent(ctx->copy_stream, ctx->consumed[k], 0);      // buffer k is free again
        if (e == cudaSuccess && fbytes)
            e = cudaMemcpyAsync(ctx->d_chunk[k], (const char*)coords + (size_t)f0 * fbytes, (size_t)nf * fbytes,
                                cudaMemcpyHostToDevice, ctx->copy_stream);               // each frame is copied once
        if (e == cudaSuccess) e = cudaEventRecord(ctx->copied[k], ctx->copy_stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, ctx->copied[k], 0);
        if (e != cudaSuccess) { rc = cuda_fail(ctx, e, "cdh_histograms_stream: copy pipeline"); break; }
        ctx->flags = c == 0 ? (saved_flags & ~CDH_FLAG_ACCUMULATE) : (saved_flags | CDH_FLAG_ACCUMULATE);
        rc = cdh_histograms(ctx, ctx->d_chunk[k], nf, off, n_species, box_type,
                            (box && n_boxes > 1) ? box + (size_t)f0 * 9 : box, n_boxes > 1 ? nf : n_boxes,
                            r_max, n_bins, precision, stream_, (uint64_t*)ctx->d_io_out);
        if (rc == CDH_OK && (e = cudaEventRecord(ctx->consumed[k], stream)) != cudaSuccess)
            rc = cuda_fail(ctx, e, "cudaEventRecord");
    }
    ctx->flags = saved_flags;
    if (rc != CDH_OK) {                     // leave nothing in flight that still reads the caller's buffer
        cudaStreamSynchronize(ctx->copy_stream); cudaStreamSynchronize(stream); cudaGetLastError();
        return rc;
    }
    CDH_CUDA(cudaMemcpyAsync(out, ctx->d_io_out, obytes, cudaMemcpyDeviceToHost, stream));
    CDH_CUDA(cudaStreamSynchronize(stream));
    return CDH_OK;
}

extern "C" int cdh_rdf(cdh_ctx* ctx, const uint64_t* hist, int32_t n_hist, int32_t n_bins, double r_max, int32_t n_frames,
                       const double* n_pairs, double volume, void* stream_, double* g) {
    if (!ctx || !hist || !n_pairs || !g || n_hist < 1 || n_bins < 1 || n_frames < 1) return CDH_ERR_INVALID_ARG;
    if (!(r_max > 0.0) || !std::isfinite(r_max) || !(volume > 0.0) || !std::isfinite(volume)) return CDH_ERR_INVALID_ARG;
    for (int h = 0; h < n_hist; ++h) if (!(n_pairs[h] >= 0.0) || !std::isfinite(n_pairs[h])) return CDH_ERR_INVALID_ARG;
    cudaStream_t stream = (cudaStream_t)stream_;
    ctx->err.clear();
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");
    int rc;
    const size_t bytes = (size_t)n_hist * sizeof(double);
    if (ctx->staged_pending) { CDH_CUDA(cudaEventSynchronize(ctx->staged)); ctx->staged_pending = false; }
    if ((rc = grow(ctx, &ctx->h_tables, &ctx->h_tables_bytes, bytes, true)) != CDH_OK) return rc;
    if ((rc = grow(ctx, &ctx->d_small, &ctx->small_bytes, bytes, false)) != CDH_OK) return rc;
    double* hd = (double*)ctx->h_tables;
    for (int h = 0; h < n_hist; ++h) hd[h] = n_pairs[h] / volume;
    CDH_CUDA(cudaMemcpyAsync(ctx->d_small, hd, bytes, cudaMemcpyHostToDevice, stream));
    CDH_CUDA(cudaEventRecord(ctx->staged, stream));
    ctx->staged_pending = true;
    RdfParams rp;
    rp.hist = (const unsigned long long*)hist; rp.density = (const double*)ctx->d_small; rp.g = g;
    rp.dr = r_max / (double)n_bins; rp.n_frames = (double)n_frames; rp.n_bins = (uint32_t)n_bins;
    rp.total = (uint64_t)n_hist * (uint64_t)n_bins;
    const uint64_t blocks = (rp.total + 255) / 256;
    if (blocks > 0x7fffffffull) return CDH_ERR_INVALID_ARG;
    rdf_kernel<<<(unsigned)blocks, 256, 0, stream>>>(rp);
    CDH_CUDA(cudaGetLastError());
    return CDH_OK;
}

// ---- host-logic hooks (include/cdh_bench.h): no device is touched, usable on a machine without a GPU ---------------
extern "C" uint32_t cdh_host_d2_threshold_bits(float rmax) { return d2_threshold_bits(rmax); }

extern "C" int cdh_host_fused_rint_constant(float inv_l, float* inv_lf) {
    return (inv_lf && fused_rint_constant(inv_l, inv_lf)) ? 1 : 0;
}

extern "C" int64_t cdh_host_work_items(int32_t n_frames, const int32_t* off, int32_t n_species, int32_t n_bins,
                                       int32_t cap_bins, int32_t ti, int32_t tj, int64_t* items, int64_t max_items) {
    if (!off || n_frames < 1 || n_species < 1 || n_bins < 1 || cap_bins < 1 || ti < 4 || tj < (int32_t)kMinChunk ||
        tj % (int32_t)kMinChunk || (tj > kStageParticles && tj % kStageParticles) || (max_items > 0 && !items))
        return -1;
    std::vector<uint32_t> pad_off((size_t)n_species + 1);
    uint64_t slots = 0;
    for (int s = 0; s < n_species; ++s) {
        pad_off[s] = (uint32_t)slots;
        slots += ((uint64_t)(off[s + 1] - off[s]) + kPadParticles - 1) / kPadParticles * kPadParticles;
    }
    pad_off[n_species] = (uint32_t)slots;
    const SweepPlan sp = plan_sweeps((uint32_t)n_bins, (uint32_t)cap_bins);
    WorkTables wt;
    build_tables(n_frames, off, n_species, 1, (uint32_t)n_bins, sp, (uint32_t)ti, (uint32_t)tj, pad_off, (uint32_t)slots, &wt);
    // expand the rows exactly as the tile kernel does: item -> (row, j-chunk)
    int64_t n = 0;
    for (size_t r = 0; r + 1 < wt.rows.size(); ++r) {
        const Row& row = wt.rows[r];
        const Seg& seg = wt.segs[row.seg];
        const uint32_t count = wt.rows[r + 1].item_prefix - row.item_prefix;
        for (uint32_t k = 0; k < count; ++k, ++n) {
            if (n >= max_items) continue;
            const uint32_t j0 = (row.jc0 + k) * (uint32_t)tj;
            const uint32_t j1 = std::min((uint32_t)seg.nj, j0 + (uint32_t)tj);
            int64_t* it = items + 8 * n;
            it[0] = seg.hist; it[1] = seg.bin_lo; it[2] = seg.bin_cnt; it[3] = row.i0; it[4] = j0; it[5] = j1;
            it[6] = seg.same; it[7] = ((int64_t)seg.i_group << 32) | seg.j_group;
        }
    }
    return n == (int64_t)wt.n_items ? n : -2;
}
