// cdh_api.cu -- the C ABI of libcdh (include/cdh.h): context, validation, host dispatch.
// All device work of a call is enqueued on the caller's stream; cdh_histograms never synchronises.
#include <cstdio>
#include <new>
#include <string>
#include "cdh_host.h"
#include "cdh_tile.cuh"
#include "cdh_f64.cuh"
#include "cdh_rdf.cuh"

using namespace cdh;

struct cdh_ctx {
    int device = 0;
    uint32_t flags = 0;
    int n_sm = 0;
    int max_smem_optin = 0;
    // device scratch, grown on demand, never shrunk
    float* d_pk = nullptr;       size_t pk_bytes = 0;
    void* d_tables = nullptr;    size_t tables_bytes = 0;     // segs | rows | boxes | off | pad_off
    unsigned int* d_scalars = nullptr;                        // [0..2] work counters of the call's tile launches, [4..9] range keys (repack_kernel)
    void* h_tables = nullptr;    size_t h_tables_bytes = 0;   // pinned staging for d_tables
    cudaEvent_t staged = nullptr;                             // h_tables may be rewritten once this has fired
    bool staged_pending = false;
    void* d_io_coords = nullptr; size_t io_coords_bytes = 0;  // cdh_histograms_host staging
    void* d_io_out = nullptr;    size_t io_out_bytes = 0;
    // cdh_histograms_stream: two chunk buffers filled on a private copy stream while the other is being processed
    void* d_chunk[2] = {nullptr, nullptr}; size_t chunk_bytes[2] = {0, 0};
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t copied[2] = {nullptr, nullptr}, consumed[2] = {nullptr, nullptr};
    cudaEvent_t* ev = nullptr;   // CDH_FLAG_TIME_KERNELS: ring of [CDH_TIMED_CALLS][4]: call begin, tile begin, tile end, call end
    uint64_t timed_calls = 0;
    std::string err;
    int64_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

namespace {

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

int grow(cdh_ctx* ctx, void** p, size_t* have, size_t need, bool pinned_host) {
    if (need <= *have) return CDH_OK;
    if (*p) {
        // a buffer still in use by enqueued work must not be freed under it
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
static double frame_pairs(const int32_t* off, int32_t n_species) {
    double tot = 0.0;
    for (int p = 0; p < n_species; ++p) {
        const double np_ = (double)(off[p + 1] - off[p]);
        tot += 0.5 * np_ * (np_ - 1.0);
        for (int q = p + 1; q < n_species; ++q) tot += np_ * (double)(off[q + 1] - off[q]);
    }
    return tot;
}

#ifndef CDH_SKIP_EFFICIENCY
#define CDH_SKIP_EFFICIENCY 0.95  // the SKIP variants (cdh_tile.cuh) are taken when fewer than this share of the pair slots the
                                  // 1024-particle i-tiles walk are pairs of the problem (measured break-even, one species per
                                  // frame: 16,384 particles, share 0.94: +0.7 %; 24,000 particles, share 0.96: -0.4 %)
#endif
// Small species: the share of the walked pair slots (1024-particle i-tiles: whole stages on the diagonal, padded last tiles)
// that are pairs of the problem decides whether the SKIP variants of the 256-thread kernels pay.
static bool small_species(const int32_t* off, int32_t n_species) {
    const double ti256 = 256.0 * kR;
    double walked = 0.0;
    for (int p = 0; p < n_species; ++p) {                       // the count build_tables makes (WorkTables::padded_pairs)
        const double np_ = (double)(off[p + 1] - off[p]), tiles = std::ceil(np_ / ti256);
        walked += ti256 * (tiles * np_ - ti256 * 0.5 * tiles * (tiles - 1.0));          // i-tile t walks j from t * 1024 to n_p
        for (int q = p + 1; q < n_species; ++q) walked += tiles * ti256 * (double)(off[q + 1] - off[q]);
    }
    return walked > 0.0 && frame_pairs(off, n_species) < CDH_SKIP_EFFICIENCY * walked;
}

// ---- kernel table -----------------------------------------------------------------------------
typedef void (*TileFn)(const TileParams);
struct Variant { TileFn fn; int threads; };

#ifndef CDH_GLOBAL_SWEEPS
#define CDH_GLOBAL_SWEEPS 8   // shared-memory sweeps from which the global-histogram mode takes over (measured
                              // break-even: 200,000 uniform points, 400,000 bins: 8 sweeps 200 vs global 221 Gpairs/s)
#endif
constexpr uint32_t kGlobalSweeps = CDH_GLOBAL_SWEEPS;
#ifndef CDH_ITEMS_PER_CTA
#define CDH_ITEMS_PER_CTA 64   // work items per resident CTA the j-chunk size is shrunk for (tail of the dynamic schedule)
#endif
constexpr uint64_t kItemsPerCta = CDH_ITEMS_PER_CTA;
#ifndef CDH_MINB
#define CDH_MINB 3      // resident CTAs per SM the 256-thread NONE / ORTHO fast variants are register-bounded for
                        // (80 registers; measured +1.5 % over 2; the triclinic variants need 128 registers: 2)
#endif
#ifndef CDH_BIG_T
#define CDH_BIG_T 1024  // threads of the one-CTA-per-SM variants (32 warps/SM: config 5 +5 % over 512)
#endif
template <int BOX, int TRI, int MODE>
Variant fast_variant(bool big, bool skip) {
    if constexpr (MODE != MODE_GLOBAL)
        if (big) return {tile_kernel<BOX, TRI, CDH_BIG_T, VAR_FAST, MODE, 1>, CDH_BIG_T};
    if constexpr (MODE == MODE_SHARED)
        if (skip) return {tile_kernel<BOX, TRI, 256, VAR_FAST, MODE, (BOX == BOX_TRI ? 2 : CDH_MINB), true>, 256};
    return {tile_kernel<BOX, TRI, 256, VAR_FAST, MODE, (BOX == BOX_TRI ? 2 : CDH_MINB)>, 256};
}
template <int SPLIT>
Variant pick_fast(int box_type, int tri, bool big, bool skip) {      // tri: TRI_* for TRICLINIC, ORTHO_* for ORTHO
    if (box_type == CDH_BOX_NONE) return fast_variant<BOX_NONE, 0, SPLIT>(big, skip);
    if (box_type == CDH_BOX_ORTHO)
        return tri == ORTHO_FUSED ? fast_variant<BOX_ORTHO, ORTHO_FUSED, SPLIT>(big, skip)
             : tri == ORTHO_EXACT ? fast_variant<BOX_ORTHO, ORTHO_EXACT, SPLIT>(big, skip) : fast_variant<BOX_ORTHO, ORTHO_PLAIN, SPLIT>(big, skip);
    if (tri == TRI_UPPER_B01) return fast_variant<BOX_TRI, TRI_UPPER_B01, SPLIT>(big, skip);
    if (tri == TRI_UPPER) return fast_variant<BOX_TRI, TRI_UPPER, SPLIT>(big, skip);
    if (tri == (TRI_UPPER_B01 | TRI_WIDE)) return fast_variant<BOX_TRI, TRI_UPPER_B01 | TRI_WIDE, SPLIT>(big, skip);
    if (tri == (TRI_UPPER | TRI_WIDE)) return fast_variant<BOX_TRI, TRI_UPPER | TRI_WIDE, SPLIT>(big, skip);
    if (tri == (TRI_GENERAL | TRI_WIDE)) return fast_variant<BOX_TRI, TRI_GENERAL | TRI_WIDE, SPLIT>(big, skip);
    return fast_variant<BOX_TRI, TRI_GENERAL, SPLIT>(big, skip);
}
template <int VAR>
Variant simple_variant(int box_type, bool big) {
    if (box_type == CDH_BOX_NONE)
        return big ? Variant{tile_kernel<BOX_NONE, 0, CDH_BIG_T, VAR, MODE_SPLIT, 1>, CDH_BIG_T} : Variant{tile_kernel<BOX_NONE, 0, 256, VAR, MODE_SPLIT, 2>, 256};
    if (box_type == CDH_BOX_ORTHO)
        return big ? Variant{tile_kernel<BOX_ORTHO, 0, CDH_BIG_T, VAR, MODE_SPLIT, 1>, CDH_BIG_T} : Variant{tile_kernel<BOX_ORTHO, 0, 256, VAR, MODE_SPLIT, 2>, 256};
    return big ? Variant{tile_kernel<BOX_TRI, 0, CDH_BIG_T, VAR, MODE_SPLIT, 1>, CDH_BIG_T} : Variant{tile_kernel<BOX_TRI, 0, 256, VAR, MODE_SPLIT, 2>, 256};
}
Variant simple_global(int box_type) {
    if (box_type == CDH_BOX_NONE) return {tile_kernel<BOX_NONE, 0, 256, VAR_SIMPLE, MODE_GLOBAL, 2>, 256};
    if (box_type == CDH_BOX_ORTHO) return {tile_kernel<BOX_ORTHO, 0, 256, VAR_SIMPLE, MODE_GLOBAL, 2>, 256};
    return {tile_kernel<BOX_TRI, 0, 256, VAR_SIMPLE, MODE_GLOBAL, 2>, 256};
}
Variant pick_simple(int box_type, bool big, uint32_t flags) {
    if (flags & CDH_FLAG_WARP_AGGREGATE) return simple_variant<VAR_SIMPLE_MATCH>(box_type, big);
    if (flags & CDH_FLAG_NO_AGGREGATE) return simple_variant<VAR_SIMPLE_PLAIN>(box_type, big);
    return simple_variant<VAR_SIMPLE>(box_type, big);
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
    if (!g.ok || cudaMalloc(&ctx->d_scalars, 64) != cudaSuccess ||
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
    if (ctx->d_pk) cudaFree(ctx->d_pk);
    if (ctx->d_tables) cudaFree(ctx->d_tables);
    if (ctx->d_scalars) cudaFree(ctx->d_scalars);
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

// ---- the double-precision call (cdh_f64.cuh): same layout, tables and stream discipline as the fp32 call --------
typedef void (*TileFn64)(const TileParams64);
static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static int histograms_f64(cdh_ctx* ctx, const double* coords, int32_t n_frames, const int32_t* off, int32_t n_species,
                          int32_t box_type, const double* box, int32_t n_boxes, double r_max, int32_t n_bins,
                          cudaStream_t stream, uint64_t* out) {
    const int nb = (box_type == CDH_BOX_NONE) ? 0 : n_boxes;
    std::vector<BoxConst64> boxes((size_t)(nb > 0 ? nb : 1));
    std::memset(boxes.data(), 0, boxes.size() * sizeof(BoxConst64));
    for (int b = 0; b < nb; ++b) {
        if (!make_box_const64(box_type, box + 9 * (size_t)b, r_max, &boxes[b])) return CDH_ERR_INVALID_ARG;
        if (ctx->flags & CDH_FLAG_NO_PRUNE) boxes[b].prune_ok = 0.0;
    }
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
    const int n_hist = n_species * (n_species + 1) / 2;

    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");

    uint32_t cap_bins = (uint32_t)((ctx->max_smem_optin - tile_smem_bytes64(0)) / 4);
    const uint32_t flag_cap = ctx->flags >> CDH_FLAG_MAX_SMEM_BINS_SHIFT;
    if (flag_cap && flag_cap < cap_bins) cap_bins = flag_cap;
    SweepPlan sp = plan_sweeps((uint32_t)n_bins, cap_bins);
    const bool global_hist = (ctx->flags & CDH_FLAG_GLOBAL_HIST) != 0 || (!flag_cap && sp.n_sweeps >= kGlobalSweeps);
    if (global_hist) { sp.n_sweeps = 1; sp.bins_per_sweep = (uint32_t)n_bins; }
    const int smem_bytes = tile_smem_bytes64(global_hist ? 0 : (int)sp.bins_per_sweep);
    const bool big = 2 * (smem_bytes + 1024) > 228 * 1024;
    TileFn64 fn; int threads;
    const bool pbox = box_type == CDH_BOX_TRICLINIC && nb == 1;      // one box: constants through the parameter bank
    const bool skip = !big && !global_hist && sp.n_sweeps == 1 && small_species(off, n_species);
    auto pick64 = [&](auto mode_c) -> TileFn64 {
        constexpr int M = decltype(mode_c)::value;
        if constexpr (M == MODE_SHARED)
            if (skip) {
                if (box_type == CDH_BOX_NONE) return tile_kernel_f64<BOX_NONE, 256, 2, false, M, true>;
                if (box_type == CDH_BOX_ORTHO) return tile_kernel_f64<BOX_ORTHO, 256, 2, false, M, true>;
                return pbox ? tile_kernel_f64<BOX_TRI, 256, 2, true, M, true> : tile_kernel_f64<BOX_TRI, 256, 2, false, M, true>;
            }
        if (box_type == CDH_BOX_NONE) return big ? tile_kernel_f64<BOX_NONE, 512, 1, false, M> : tile_kernel_f64<BOX_NONE, 256, 2, false, M>;
        if (box_type == CDH_BOX_ORTHO) return big ? tile_kernel_f64<BOX_ORTHO, 512, 1, false, M> : tile_kernel_f64<BOX_ORTHO, 256, 2, false, M>;
        if (pbox) return big ? tile_kernel_f64<BOX_TRI, 512, 1, true, M> : tile_kernel_f64<BOX_TRI, 256, 2, true, M>;
        return big ? tile_kernel_f64<BOX_TRI, 512, 1, false, M> : tile_kernel_f64<BOX_TRI, 256, 2, false, M>;
    };
    fn = global_hist ? pick64(std::integral_constant<int, MODE_GLOBAL>{})
       : sp.n_sweeps > 1 ? pick64(std::integral_constant<int, MODE_SPLIT>{}) : pick64(std::integral_constant<int, MODE_SHARED>{});
    threads = big ? 512 : 256;
    const uint32_t ti = (uint32_t)threads * kR;
    CDH_CUDA(cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    int resident = 0;
    CDH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, (const void*)fn, threads, (size_t)smem_bytes));
    if (resident < 1) resident = 1;
    const uint32_t grid_full = (uint32_t)ctx->n_sm * (uint32_t)resident;

    WorkTables wt;
    uint32_t tj = 8192;
    for (;; tj >>= 1) {
        build_tables(n_frames, off, n_species, nb > 0 ? nb : 1, (uint32_t)n_bins, sp, ti, tj, pad_off, frame_slots, &wt);
        if (wt.n_items >= kItemsPerCta * grid_full || tj == (uint32_t)kStageParticles) break;
    }
    if (wt.n_items >= 0xffffffffull || wt.rows.size() >= 0x7fffffffull) return CDH_ERR_INVALID_ARG;

    const size_t b_segs = align256(wt.segs.size() * sizeof(Seg) + 1), b_rows = align256(wt.rows.size() * sizeof(Row)),
                 b_boxes = align256(boxes.size() * sizeof(BoxConst64)), b_off = align256(((size_t)n_species + 1) * 4);
    const size_t tables = b_segs + b_rows + b_boxes + 2 * b_off;
    int rc;
    if (ctx->staged_pending) { CDH_CUDA(cudaEventSynchronize(ctx->staged)); ctx->staged_pending = false; }
    if ((rc = grow(ctx, &ctx->h_tables, &ctx->h_tables_bytes, tables, true)) != CDH_OK) return rc;
    if ((rc = grow(ctx, &ctx->d_tables, &ctx->tables_bytes, tables, false)) != CDH_OK) return rc;
    const size_t pk_need = (size_t)n_frames * frame_slots * 3 * sizeof(double);
    if ((rc = grow(ctx, (void**)&ctx->d_pk, &ctx->pk_bytes, pk_need > 0 ? pk_need : 16, false)) != CDH_OK) return rc;

    char* h = (char*)ctx->h_tables;
    std::memcpy(h, wt.segs.data(), wt.segs.size() * sizeof(Seg));
    std::memcpy(h + b_segs, wt.rows.data(), wt.rows.size() * sizeof(Row));
    std::memcpy(h + b_segs + b_rows, boxes.data(), boxes.size() * sizeof(BoxConst64));
    std::memcpy(h + b_segs + b_rows + b_boxes, off, ((size_t)n_species + 1) * 4);
    std::memcpy(h + b_segs + b_rows + b_boxes + b_off, pad_off.data(), ((size_t)n_species + 1) * 4);
    char* d = (char*)ctx->d_tables;
    const bool timing = ctx->ev != nullptr;
    cudaEvent_t* ev = timing ? ctx->ev + 4 * (ctx->timed_calls % CDH_TIMED_CALLS) : nullptr;
    if (timing) CDH_CUDA(cudaEventRecord(ev[0], stream));
    CDH_CUDA(cudaMemcpyAsync(d, h, tables, cudaMemcpyHostToDevice, stream));
    CDH_CUDA(cudaEventRecord(ctx->staged, stream));
    ctx->staged_pending = true;
    CDH_CUDA(cudaMemsetAsync(ctx->d_scalars, 0, 64, stream));
    if (!(ctx->flags & CDH_FLAG_ACCUMULATE))
        CDH_CUDA(cudaMemsetAsync(out, 0, (size_t)n_hist * (size_t)n_bins * sizeof(uint64_t), stream));

    int launches = 0;
    if (frame_slots > 0) {
        RepackParams64 rp;
        rp.coords = coords; rp.pk = (double*)ctx->d_pk;
        rp.off = (const int32_t*)(d + b_segs + b_rows + b_boxes);
        rp.pad_off = (const uint32_t*)(d + b_segs + b_rows + b_boxes + b_off);
        rp.range_keys = ctx->d_scalars + 4;
        rp.boxes = (const BoxConst64*)(d + b_segs + b_rows);
        rp.n_species = n_species; rp.n_total = off[n_species]; rp.n_frames = n_frames;
        rp.box_type = box_type; rp.n_boxes = nb > 0 ? nb : 1;
        rp.frame_slots = frame_slots; rp.blocks_per_frame = (frame_slots + 255) / 256;
        const uint64_t blocks = (uint64_t)rp.blocks_per_frame * (uint64_t)n_frames;
        if (blocks > 0x7fffffffull) return CDH_ERR_INVALID_ARG;
        repack_kernel_f64<<<(unsigned)blocks, 256, 0, stream>>>(rp);
        CDH_CUDA(cudaGetLastError());
        ++launches;
    }
    uint32_t grid = 0;
    if (timing) CDH_CUDA(cudaEventRecord(ev[1], stream));
    if (wt.n_items > 0) {
        TileParams64 tp;
        tp.pk = (const double*)ctx->d_pk; tp.segs = (const Seg*)d; tp.rows = (const Row*)(d + b_segs);
        tp.boxes = (const BoxConst64*)(d + b_segs + b_rows);
        tp.counter = ctx->d_scalars; tp.out = (unsigned long long*)out; tp.range_keys = ctx->d_scalars + 4;
        tp.n_rows = (uint32_t)wt.rows.size() - 1; tp.n_items = (uint32_t)wt.n_items;
        tp.n_bins = (uint32_t)n_bins; tp.tj = tj; tp.smem_bins = global_hist ? 0u : sp.bins_per_sweep;
        tp.rmax = r_max; tp.scale = (double)n_bins / r_max;
        tp.box0 = boxes[0];
        grid = grid_full < tp.n_items ? grid_full : tp.n_items;
        fn<<<grid, threads, smem_bytes, stream>>>(tp);
        CDH_CUDA(cudaGetLastError());
        ++launches;
    }
    if (timing) {
        CDH_CUDA(cudaEventRecord(ev[2], stream));
        CDH_CUDA(cudaEventRecord(ev[3], stream));
        ++ctx->timed_calls;
    }
    ctx->info[0] = launches; ctx->info[1] = (int64_t)wt.n_items; ctx->info[2] = sp.n_sweeps; ctx->info[3] = grid;
    ctx->info[4] = threads; ctx->info[5] = smem_bytes;
    ctx->info[6] = 2 | ((int)global_hist << 2) | (box_type << 4) | ((int)(sp.n_sweeps > 1) << 12) | ((int)big << 13) | ((int)skip << 14) |
                   ((int64_t)tj << 16);
    ctx->info[7] = (int64_t)wt.padded_pairs;
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
    if (!((float)r_max > 0.0f) || !std::isfinite((float)r_max)) return CDH_ERR_INVALID_ARG;
    const float scale = (float)((double)n_bins / r_max);
    if (!std::isfinite(scale) || !(scale > 0.0f)) return CDH_ERR_INVALID_ARG;
    return CDH_OK;
}

extern "C" int cdh_histograms(cdh_ctx* ctx, const void* coords, int32_t n_frames, const int32_t* off,
                              int32_t n_species, int32_t box_type, const double* box, int32_t n_boxes,
                              double r_max, int32_t n_bins, int32_t precision, void* stream_, uint64_t* out) {
    if (!ctx) return CDH_ERR_INVALID_ARG;
    int rc = validate(coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, precision, out);
    if (rc != CDH_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    ctx->err.clear();
    // the double-precision kernels bin sqrt(d2) < 2^-485 as 0: harmless while it lands in bin 0 and is kept
    if (precision == CDH_F64 && !(r_max > 1e-100 && (double)n_bins / r_max < 1e100)) return CDH_ERR_INVALID_ARG;
    if (precision == CDH_F64)
        return histograms_f64(ctx, (const double*)coords, n_frames, off, n_species, box_type, box, n_boxes, r_max, n_bins, stream, out);

    // ---- host-derived constants ----------------------------------------------------------------
    const int nb = (box_type == CDH_BOX_NONE) ? 0 : n_boxes;
    std::vector<BoxConst> boxes((size_t)(nb > 0 ? nb : 1));
    std::memset(boxes.data(), 0, boxes.size() * sizeof(BoxConst));
    for (int b = 0; b < nb; ++b) {
        if (!make_box_const(box_type, box + 9 * (size_t)b, r_max, &boxes[b])) return CDH_ERR_INVALID_ARG;
        if (ctx->flags & CDH_FLAG_NO_PRUNE) boxes[b].prune_ok = 0.0f;
    }
    const int tri = (box_type == CDH_BOX_TRICLINIC) ? tri_kind(boxes.data(), nb) : 0;
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
    const int n_hist = n_species * (n_species + 1) / 2;

    DeviceGuard guard(ctx->device);
    if (!guard.ok) return cuda_fail(ctx, cudaGetLastError(), "cudaSetDevice");

    // ---- variant, sweeps, tile sizes -----------------------------------------------------------
    uint32_t cap_bins = (uint32_t)((ctx->max_smem_optin - tile_smem_bytes(0)) / 4);
    const uint32_t flag_cap = ctx->flags >> CDH_FLAG_MAX_SMEM_BINS_SHIFT;
    if (flag_cap && flag_cap < cap_bins) cap_bins = flag_cap;
    SweepPlan sp = plan_sweeps((uint32_t)n_bins, cap_bins);
    // Very wide histograms (the paper's global-memory kernel regime): beyond kGlobalSweeps
    // sweeps the private copy is dropped and updates go straight to the uint64 result in L2 (MODE_GLOBAL).
    const bool global_hist = (ctx->flags & CDH_FLAG_GLOBAL_HIST) != 0 || (!flag_cap && sp.n_sweeps >= kGlobalSweeps);
    if (global_hist) { sp.n_sweeps = 1; sp.bins_per_sweep = (uint32_t)n_bins; }
    const int smem_bytes = tile_smem_bytes(global_hist ? 0 : (int)sp.bins_per_sweep);
    const bool big = 2 * (smem_bytes + 1024) > 228 * 1024;          // one CTA per SM
    const bool split = sp.n_sweeps > 1;
    const bool use_simple_only = (ctx->flags & (CDH_FLAG_SIMPLE_KERNEL | CDH_FLAG_WARP_AGGREGATE | CDH_FLAG_NO_AGGREGATE)) != 0 ||
                                 !(scale_f < 5.0e14f);
    // Launch plan: every tile launch of the call owns an interval (lo, hi] of the fractional-coordinate range the
    // repack kernel measures, and exactly one of them does the work (cdh_tile.cuh).
    //   ORTHO: fused rint up to 1.49 (exact-product form if the host found no fused constants for some box),
    //          magic-number rint up to 2^20, library rintf beyond;  TRICLINIC: fast path up to 1.49 (n in {-1,0,1}), wide fast path up to 64,
    //          definition beyond.
    struct Launch { Variant v; float lo, hi; };
    const float kInf = INFINITY, kSmall = 1.49f, kWide = 64.0f, kMagic = 1048576.0f;
    bool fused_ok = box_type == CDH_BOX_ORTHO;
    for (int b = 0; b < nb && fused_ok; ++b) fused_ok = boxes[b].prune_ok != 0.0f;
    if (ctx->flags & CDH_FLAG_NO_PRUNE) fused_ok = false;          // tests: force the plain magic-number form
    const bool skip = small_species(off, n_species);
    auto fast_of = [&](int form) {
        return global_hist ? pick_fast<MODE_GLOBAL>(box_type, form, big, false)
                           : split ? pick_fast<MODE_SPLIT>(box_type, form, big, false) : pick_fast<MODE_SHARED>(box_type, form, big, skip);
    };
    const Variant vs = global_hist ? simple_global(box_type) : pick_simple(box_type, big, ctx->flags);
    std::vector<Launch> plan;
    if (use_simple_only) plan.push_back({vs, -kInf, kInf});
    else if (box_type == CDH_BOX_NONE) plan.push_back({fast_of(0), -kInf, kInf});
    else if (box_type == CDH_BOX_ORTHO) {
        const bool plain_only = (ctx->flags & CDH_FLAG_NO_PRUNE) != 0;     // tests: the pinned 5-operation form everywhere
        if (plain_only) plan.push_back({fast_of(ORTHO_PLAIN), -kInf, kMagic});
        else { plan.push_back({fast_of(fused_ok ? ORTHO_FUSED : ORTHO_EXACT), -kInf, kSmall}); plan.push_back({fast_of(ORTHO_PLAIN), kSmall, kMagic}); }
        plan.push_back({vs, kMagic, kInf});
    } else {
        plan.push_back({fast_of(tri), -kInf, kSmall});
        plan.push_back({fast_of(tri | TRI_WIDE), kSmall, kWide});      // unwrapped coordinates, up to 64 cells
        plan.push_back({vs, kWide, kInf});
    }
    const Variant vf = plan[0].v;
    const uint32_t ti = (uint32_t)vf.threads * kR;
    CDH_CUDA(cudaFuncSetAttribute((const void*)vf.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    int resident = 0;      // CTAs of the production variant that fit one SM (registers, shared memory)
    CDH_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, (const void*)vf.fn, vf.threads, (size_t)smem_bytes));
    if (resident < 1) resident = 1;
    const uint32_t grid_full = (uint32_t)ctx->n_sm * (uint32_t)resident;

    WorkTables wt;
    uint32_t tj = 8192;
    for (;; tj >>= 1) {
        build_tables(n_frames, off, n_species, nb > 0 ? nb : 1, (uint32_t)n_bins, sp, ti, tj, pad_off, frame_slots, &wt);
        if (wt.n_items >= kItemsPerCta * grid_full || tj == (uint32_t)kStageParticles) break;
    }
    if (wt.n_items >= 0xffffffffull || wt.rows.size() >= 0x7fffffffull) return CDH_ERR_INVALID_ARG;

    // ---- scratch -------------------------------------------------------------------------------
    const size_t b_segs = align256(wt.segs.size() * sizeof(Seg) + 1), b_rows = align256(wt.rows.size() * sizeof(Row)),
                 b_boxes = align256(boxes.size() * sizeof(BoxConst)), b_off = align256(((size_t)n_species + 1) * 4);
    const size_t tables = b_segs + b_rows + b_boxes + 2 * b_off;
    if (ctx->staged_pending) { CDH_CUDA(cudaEventSynchronize(ctx->staged)); ctx->staged_pending = false; }
    if ((rc = grow(ctx, &ctx->h_tables, &ctx->h_tables_bytes, tables, true)) != CDH_OK) return rc;
    if ((rc = grow(ctx, &ctx->d_tables, &ctx->tables_bytes, tables, false)) != CDH_OK) return rc;
    const size_t pk_need = (size_t)n_frames * frame_slots * 3 * sizeof(float);
    if ((rc = grow(ctx, (void**)&ctx->d_pk, &ctx->pk_bytes, pk_need > 0 ? pk_need : 16, false)) != CDH_OK) return rc;

    char* h = (char*)ctx->h_tables;
    std::memcpy(h, wt.segs.data(), wt.segs.size() * sizeof(Seg));
    std::memcpy(h + b_segs, wt.rows.data(), wt.rows.size() * sizeof(Row));
    std::memcpy(h + b_segs + b_rows, boxes.data(), boxes.size() * sizeof(BoxConst));
    std::memcpy(h + b_segs + b_rows + b_boxes, off, ((size_t)n_species + 1) * 4);
    std::memcpy(h + b_segs + b_rows + b_boxes + b_off, pad_off.data(), ((size_t)n_species + 1) * 4);
    char* d = (char*)ctx->d_tables;
    const bool timing = ctx->ev != nullptr;
    cudaEvent_t* ev = timing ? ctx->ev + 4 * (ctx->timed_calls % CDH_TIMED_CALLS) : nullptr;
    if (timing) CDH_CUDA(cudaEventRecord(ev[0], stream));
    CDH_CUDA(cudaMemcpyAsync(d, h, tables, cudaMemcpyHostToDevice, stream));
    CDH_CUDA(cudaEventRecord(ctx->staged, stream));
    ctx->staged_pending = true;
    CDH_CUDA(cudaMemsetAsync(ctx->d_scalars, 0, 64, stream));
    if (!(ctx->flags & CDH_FLAG_ACCUMULATE))
        CDH_CUDA(cudaMemsetAsync(out, 0, (size_t)n_hist * (size_t)n_bins * sizeof(uint64_t), stream));

    int launches = 0;
    // ---- K0 repack -----------------------------------------------------------------------------
    if (frame_slots > 0) {
        RepackParams rp;
        rp.coords = (const float*)coords; rp.pk = ctx->d_pk;
        rp.off = (const int32_t*)(d + b_segs + b_rows + b_boxes);
        rp.pad_off = (const uint32_t*)(d + b_segs + b_rows + b_boxes + b_off);
        rp.range_keys = ctx->d_scalars + 4;
        rp.boxes = (const BoxConst*)(d + b_segs + b_rows);
        rp.n_species = n_species; rp.n_total = off[n_species]; rp.n_frames = n_frames;
        rp.box_type = box_type; rp.n_boxes = nb > 0 ? nb : 1;
        rp.frame_slots = frame_slots; rp.blocks_per_frame = (frame_slots + 255) / 256;
        const uint64_t blocks = (uint64_t)rp.blocks_per_frame * (uint64_t)n_frames;
        if (blocks > 0x7fffffffull) return CDH_ERR_INVALID_ARG;
        repack_kernel<<<(unsigned)blocks, 256, 0, stream>>>(rp);
        CDH_CUDA(cudaGetLastError());
        ++launches;
    }

    // ---- K1 tile kernel(s) ---------------------------------------------------------------------
    uint32_t grid = 0;
    if (timing) CDH_CUDA(cudaEventRecord(ev[1], stream));
    if (wt.n_items > 0) {
        TileParams tp;
        tp.pk = ctx->d_pk; tp.segs = (const Seg*)d; tp.rows = (const Row*)(d + b_segs);
        tp.boxes = (const BoxConst*)(d + b_segs + b_rows);
        tp.out = (unsigned long long*)out; tp.range_keys = ctx->d_scalars + 4;
        tp.n_rows = (uint32_t)wt.rows.size() - 1; tp.n_items = (uint32_t)wt.n_items;
        tp.n_bins = (uint32_t)n_bins; tp.tj = tj; tp.smem_bins = global_hist ? 0u : sp.bins_per_sweep;
        tp.rmax = rmax_f; tp.scale = scale_f; tp.thr2_bits = d2_threshold_bits(rmax_f); tp.one = 1.0f;
        grid = grid_full < tp.n_items ? grid_full : tp.n_items;
        for (size_t k = 0; k < plan.size(); ++k) {
            tp.counter = ctx->d_scalars + k;
            tp.range_lo = plan[k].lo; tp.range_hi = plan[k].hi;
            if (k > 0) CDH_CUDA(cudaFuncSetAttribute((const void*)plan[k].v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
            plan[k].v.fn<<<grid, plan[k].v.threads, smem_bytes, stream>>>(tp);
            CDH_CUDA(cudaGetLastError());
            ++launches;
        }
    }
    if (timing) {
        CDH_CUDA(cudaEventRecord(ev[2], stream));
        CDH_CUDA(cudaEventRecord(ev[3], stream));
        ++ctx->timed_calls;
    }
    ctx->info[0] = launches; ctx->info[1] = (int64_t)wt.n_items; ctx->info[2] = sp.n_sweeps; ctx->info[3] = grid;
    ctx->info[4] = vf.threads; ctx->info[5] = smem_bytes;
    const int form = box_type == CDH_BOX_ORTHO ? ((ctx->flags & CDH_FLAG_NO_PRUNE) ? ORTHO_PLAIN : fused_ok ? ORTHO_FUSED : ORTHO_EXACT) : tri;
    const bool skip_used = skip && !big && !split && !global_hist && !use_simple_only;
    ctx->info[6] = (use_simple_only ? 0 : 1) | ((int)global_hist << 2) | (box_type << 4) | (form << 8) | ((int)split << 12) | ((int)big << 13) |
                   ((int)skip_used << 14) | ((int64_t)tj << 16);
    ctx->info[7] = (int64_t)wt.padded_pairs;
    return CDH_OK;
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
    if ((rc = grow(ctx, &ctx->d_tables, &ctx->tables_bytes, bytes, false)) != CDH_OK) return rc;
    double* hd = (double*)ctx->h_tables;
    for (int h = 0; h < n_hist; ++h) hd[h] = n_pairs[h] / volume;
    CDH_CUDA(cudaMemcpyAsync(ctx->d_tables, hd, bytes, cudaMemcpyHostToDevice, stream));
    CDH_CUDA(cudaEventRecord(ctx->staged, stream));
    ctx->staged_pending = true;
    RdfParams rp;
    rp.hist = (const unsigned long long*)hist; rp.density = (const double*)ctx->d_tables; rp.g = g;
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
    if (!off || n_frames < 1 || n_species < 1 || n_bins < 1 || cap_bins < 1 || ti < 4 || tj < kStageParticles ||
        tj % kStageParticles || (max_items > 0 && !items))
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
