// cdh_noalloc.cu -- cdh_histograms_noalloc (include/cdh.h): the histogram call for callers that must not allocate.
//
// Every other entry point keeps its device scratch (repacked coordinates, work tables, work counters) in buffers a
// context obtained from cudaMalloc / cudaMallocHost.  Code under CUDA graph capture, tight serving loops and harnesses
// that forbid allocation cannot create a context.  This entry point needs none: its scratch is ONE file-scope device
// array of a fixed, modest size (kScratchBytes, 1.75 MiB) that every GPU holds from the moment it loads the library.
// The call enqueues the same kernels as the context path -- K0 repack_kernel and ONE K1 tile_kernel launch
// (cdh_kernels.cuh, cdh_sched.cuh) -- with every scratch pointer aimed into that array, and calls no cudaMalloc,
// cudaFree, cudaMallocHost or other allocating CUDA routine; the work tables go up with one cudaMemcpyAsync from
// pageable host memory (the driver stages it; the host vectors may die when the call returns).
//
// Kernel variants: no box -> the production packed-fp32 kernel (MathFast<BOX_NONE>); periodic boxes -> the plain
// cross-validation kernel (MathSimple, library sqrtf / rintf / floorf, exact for any coordinate range), which needs no
// host-searched constants and no launch gates.  Both return the integers of the pinned sequence, i.e. the
// same result as cdh_histograms.
//
// The array is shared by every call on the device and keeps the last call's contents.  What must start at zero (work
// counter, range keys, the caller's result) is cleared by the call itself; the repacked coordinates and the tables are
// rewritten completely.  Two calls that overlap on one GPU (different streams, different host threads) RACE on the
// array: callers serialise them (one stream, or events).  Recording into a CUDA graph: calls whose work tables fit a kernel
// parameter (32,000 bytes: e.g. 3 species x 100 frames, or one frame of any size the scratch holds) have no node that reads
// host memory and can be replayed; larger ones are refused on a capturing stream.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>
#include "cdh_host.h"
#include "cdh_math32.cuh"
#include "cdh_variants.h"

using namespace cdh;

namespace {

constexpr size_t kMaxSlots = CDH_NOALLOC_MAX_PADDED_PARTICLES;     // padded particles over all frames (species padded to 4096)
constexpr size_t kScalarBytes = 256;                               // [0,64) counters + range keys | [64,128) the repack kernel's "next set"
constexpr size_t kTableBytes = 262144 - kScalarBytes;              // segs | rows | boxes | off | pad_off
constexpr size_t kPkBytes = kMaxSlots * 3 * sizeof(float);
constexpr size_t kScratchBytes = kScalarBytes + kTableBytes + kPkBytes;
static_assert(kScratchBytes == CDH_NOALLOC_SCRATCH_BYTES, "include/cdh.h states the size of the static scratch");

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: the address the kernels get
// comes from cudaGetSymbolAddress (device_setup below), once per device, with that device current.
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
struct DeviceSetup {
    bool ready = false;
    unsigned char* scratch = nullptr;   // device address of g_scratch on this device
    int n_sm = 0, max_smem_optin = 0;
};
DeviceSetup g_dev[kMaxDevices];
std::mutex g_mutex;
thread_local std::string t_err;

int fail(int code, const std::string& what) { t_err = what; return code; }
int cuda_fail(cudaError_t e, const char* what) {
    t_err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return CDH_ERR_CUDA;
}
#define NA_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

struct DeviceGuard {
    int prev = -1; bool ok;
    explicit DeviceGuard(int dev) { ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// Once per device, with that device current (the caller holds the guard and the mutex).
int device_setup(int device, DeviceSetup** out) {
    DeviceSetup& d = g_dev[device];
    if (!d.ready) {
        int major = 0;
        NA_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device));
        if (major != 10) return fail(CDH_ERR_INVALID_ARG, "cdh_histograms_noalloc: not an sm_100 device");
        NA_CUDA(cudaDeviceGetAttribute(&d.n_sm, cudaDevAttrMultiProcessorCount, device));
        NA_CUDA(cudaDeviceGetAttribute(&d.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device));
        void* p = nullptr;
        NA_CUDA(cudaGetSymbolAddress(&p, g_scratch));
        if (!p) return fail(CDH_ERR_CUDA, "cudaGetSymbolAddress returned no address");
        d.scratch = static_cast<unsigned char*>(p);
        d.ready = true;
    }
    *out = &d;
    return CDH_OK;
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// Small work tables travel as a kernel PARAMETER (copied by value when the launch is enqueued or recorded), not as a copy from
// host memory: the call then has no node that reads the host, and can be recorded into a CUDA graph and replayed.
template <int N16>
struct alignas(16) TableBlob { uint4 q[N16]; };
constexpr int kBlobSmall = 250, kBlobLarge = 2000;            // 4,000 and 32,000 bytes (kernel parameters: up to 32,764 bytes)

template <int N16>
__global__ void __launch_bounds__(256) tables_from_params(const __grid_constant__ TableBlob<N16> blob, uint4* dst, uint32_t n16) {
    for (uint32_t k = blockIdx.x * 256u + threadIdx.x; k < n16; k += gridDim.x * 256u) dst[k] = blob.q[k];
}

template <int N16>
cudaError_t upload_by_value(const unsigned char* h, size_t bytes, unsigned char* dst, cudaStream_t stream) {
    static thread_local TableBlob<N16> blob;                   // host staging of the parameter (static: no allocation per call)
    std::memcpy(blob.q, h, bytes);
    const uint32_t n16 = (uint32_t)((bytes + 15) / 16);
    tables_from_params<N16><<<(n16 + 255) / 256, 256, 0, stream>>>(blob, reinterpret_cast<uint4*>(dst), n16);
    return cudaGetLastError();
}

}  // namespace

extern "C" const char* cdh_noalloc_last_error(void) { return t_err.c_str(); }

extern "C" int cdh_histograms_noalloc(int device, const void* coords, int32_t n_frames, const int32_t* off, int32_t n_species,
                                      int32_t box_type, const double* box, int32_t n_boxes, double r_max, int32_t n_bins,
                                      void* stream_, uint64_t* out) {
    t_err.clear();
    // ---- argument checks (as cdh_histograms, CDH_F32): nothing is enqueued on error -------------------------------
    if (!coords || !off || !out) return fail(CDH_ERR_INVALID_ARG, "null pointer");
    if (device < 0 || device >= kMaxDevices) return fail(CDH_ERR_INVALID_ARG, "no such device");
    if (n_frames < 1 || n_species < 1 || n_species > 4096 || n_bins < 1) return fail(CDH_ERR_INVALID_ARG, "n_frames / n_species / n_bins");
    if (!(r_max > 0.0) || !std::isfinite(r_max) || !((float)r_max > 0.0f) || !std::isfinite((float)r_max)) return fail(CDH_ERR_INVALID_ARG, "r_max");
    if (box_type != CDH_BOX_NONE && box_type != CDH_BOX_ORTHO && box_type != CDH_BOX_TRICLINIC) return fail(CDH_ERR_INVALID_ARG, "box_type");
    if (box_type == CDH_BOX_NONE ? (box != nullptr) : (box == nullptr)) return fail(CDH_ERR_INVALID_ARG, "box");
    if (box_type != CDH_BOX_NONE && n_boxes != 1 && n_boxes != n_frames) return fail(CDH_ERR_INVALID_ARG, "n_boxes");
    if (off[0] != 0) return fail(CDH_ERR_INVALID_ARG, "species_offsets[0] != 0");
    for (int s = 0; s < n_species; ++s) if (off[s + 1] < off[s]) return fail(CDH_ERR_INVALID_ARG, "species_offsets not ascending");
    const float rmax_f = (float)r_max, scale_f = (float)((double)n_bins / r_max);
    if (!std::isfinite(scale_f) || !(scale_f > 0.0f)) return fail(CDH_ERR_INVALID_ARG, "n_bins / r_max");
    if (n_bins > CDH_NOALLOC_MAX_BINS)
        return fail(CDH_ERR_UNSUPPORTED, "cdh_histograms_noalloc: n_bins = " + std::to_string(n_bins) + " exceeds the maximum of " +
                                             std::to_string(CDH_NOALLOC_MAX_BINS) + " (use cdh_histograms)");

    // ---- padded layout and its limit ---------------------------------------------------------------------------
    std::vector<uint32_t> pad_off((size_t)n_species + 1);
    uint64_t slots = 0;
    for (int s = 0; s < n_species; ++s) {
        pad_off[s] = (uint32_t)slots;
        const uint64_t n = (uint64_t)(off[s + 1] - off[s]);
        slots += (n + kPadParticles - 1) / kPadParticles * kPadParticles;
        if (slots > kMaxSlots) break;
    }
    if (slots * (uint64_t)n_frames > kMaxSlots)
        return fail(CDH_ERR_UNSUPPORTED, "cdh_histograms_noalloc: the call needs more than the maximum of " + std::to_string(kMaxSlots) +
                                             " padded particles (every species of every frame padded to " + std::to_string(kPadParticles) +
                                             "): use cdh_histograms");
    pad_off[n_species] = (uint32_t)slots;
    const uint32_t frame_slots = (uint32_t)slots;
    const uint32_t blocks_per_frame = (frame_slots + 255) / 256;
    const int n_hist = n_species * (n_species + 1) / 2;
    const uint64_t out_count = (uint64_t)n_hist * (uint64_t)n_bins;

    const int nb = (box_type == CDH_BOX_NONE) ? 0 : n_boxes;
    const size_t n_box_rec = (size_t)(nb > 0 ? nb : 1);
    std::vector<BoxConst> boxes(n_box_rec);
    std::memset(boxes.data(), 0, boxes.size() * sizeof(BoxConst));
    for (int b = 0; b < nb; ++b)
        if (!make_box_const(box_type, box + 9 * (size_t)b, r_max, &boxes[b])) return fail(CDH_ERR_INVALID_ARG, "box is singular or not finite");

    // ---- device set-up (once per device): the address of the static scratch -----------------------------------------
    std::lock_guard<std::mutex> lock(g_mutex);
    DeviceGuard guard(device);
    if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
    DeviceSetup* dev = nullptr;
    int rc = device_setup(device, &dev);
    if (rc != CDH_OK) return rc;
    cudaStream_t stream = (cudaStream_t)stream_;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    NA_CUDA(cudaStreamIsCapturing(stream, &cap));
    const bool capturing = cap != cudaStreamCaptureStatusNone;     // the call is being recorded into a CUDA graph
    unsigned char* const scratch = dev->scratch;
    unsigned int* const scalars = reinterpret_cast<unsigned int*>(scratch);
    unsigned char* const d_tables = scratch + kScalarBytes;
    float* const d_pk = reinterpret_cast<float*>(scratch + kScalarBytes + kTableBytes);

    // ---- kernel variant, shared memory, grid ---------------------------------------------------------------------
    const bool fast = box_type == CDH_BOX_NONE && scale_f < 5.0e14f;
    const int mode = fast ? MODE_SHARED : MODE_SPLIT;        // the plain kernels name the whole-histogram-in-shared-memory mode SPLIT (1 sweep)
    using MF = MathFast<BOX_NONE, 0>;
    const uint32_t cap_ring = (uint32_t)((dev->max_smem_optin - tile_smem_fixed<MF>(4)) / 4 - 2);
    const uint32_t cap_two = (uint32_t)((dev->max_smem_optin - tile_smem_fixed<MF>(2)) / 4 - 2);
    if ((uint32_t)n_bins > cap_two) return fail(CDH_ERR_UNSUPPORTED, "cdh_histograms_noalloc: n_bins exceeds the shared memory of one CTA");
    const int n_stages = (uint32_t)n_bins > cap_ring ? 2 : 4;
    const int smem_bytes = tile_smem_bytes<MF>(n_stages, n_bins);
    const bool big = 2 * (smem_bytes + 1024) > 228 * 1024;   // fewer than two 256-thread CTAs fit one SM: one CTA of 1,024 threads
    const int shape = big ? SHAPE_BIG : SHAPE_256;
    const Variant v = fast ? fast_variant_none(mode, shape) : simple_variant(box_type, VAR_SIMPLE, mode, shape);
    if (!v.fn) return fail(CDH_ERR_UNSUPPORTED, "kernel variant not built");
    NA_CUDA(cudaFuncSetAttribute(v.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
    int resident = 0;
    NA_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, v.fn, v.threads, (size_t)smem_bytes));
    if (resident < 1) resident = 1;
    const uint32_t grid_full = (uint32_t)dev->n_sm * (uint32_t)resident;

    // ---- work tables (host), as the context path builds them -----------------------------------------------------------
    SweepPlan sp; sp.n_sweeps = 1; sp.bins_per_sweep = (uint32_t)n_bins;
    const uint32_t ti = (uint32_t)v.threads * kR;
    WorkTables wt;
    uint32_t tj = 8192;
    for (;; tj >>= 1) {
        build_tables(n_frames, off, n_species, nb > 0 ? nb : 1, (uint32_t)n_bins, sp, ti, tj, pad_off, frame_slots, &wt);
        if (wt.n_items >= 128ull * grid_full) break;
        if (tj <= (uint32_t)kStageParticles && (wt.n_items >= grid_full || tj == 32u)) break;
    }
    if (wt.n_items >= 0xf0000000ull) return fail(CDH_ERR_INVALID_ARG, "too many work items");
    const size_t b_segs = align256(wt.segs.size() * sizeof(Seg) + 1), b_rows = align256(wt.rows.size() * sizeof(Row)),
                 b_boxes = align256(n_box_rec * sizeof(BoxConst)), b_off = align256(((size_t)n_species + 1) * 4);
    const size_t o_rows = b_segs, o_boxes = o_rows + b_rows, o_off = o_boxes + b_boxes, o_pad = o_off + b_off, tables = o_pad + b_off;
    if (tables > kTableBytes)
        return fail(CDH_ERR_UNSUPPORTED, "cdh_histograms_noalloc: the work tables of the call (" + std::to_string(tables) +
                                             " bytes: frames x species pairs x i-tiles) exceed the maximum of " + std::to_string(kTableBytes) +
                                             " bytes: use cdh_histograms");
    // Larger tables are copied from host memory that dies with this call: recorded into a graph, that copy would read freed
    // memory on every replay.  Refuse instead of corrupting.
    if (capturing && tables > (size_t)kBlobLarge * 16)
        return fail(CDH_ERR_UNSUPPORTED, "cdh_histograms_noalloc: the stream is being captured into a CUDA graph and the work tables of the call (" +
                                             std::to_string(tables) + " bytes) exceed the " + std::to_string(kBlobLarge * 16) +
                                             " bytes that travel as a kernel parameter; this call cannot be replayed (cached cdh_histograms calls can)");
    std::vector<unsigned char> h(align256(tables) + 16, 0);
    std::memcpy(h.data(), wt.segs.data(), wt.segs.size() * sizeof(Seg));
    std::memcpy(h.data() + o_rows, wt.rows.data(), wt.rows.size() * sizeof(Row));
    std::memcpy(h.data() + o_boxes, boxes.data(), n_box_rec * sizeof(BoxConst));
    std::memcpy(h.data() + o_off, off, ((size_t)n_species + 1) * 4);
    std::memcpy(h.data() + o_pad, pad_off.data(), ((size_t)n_species + 1) * 4);

    // ---- enqueue: clear what must start at zero, tables, K0 repack, K1 tile ------------------------------------------------
    NA_CUDA(cudaMemsetAsync(scalars, 0, 128, stream));                               // work counter, range keys
    NA_CUDA(cudaMemsetAsync(out, 0, out_count * sizeof(uint64_t), stream));          // the caller's result is overwritten
    if (frame_slots == 0) return CDH_OK;
    if (tables <= (size_t)kBlobSmall * 16) NA_CUDA(upload_by_value<kBlobSmall>(h.data(), tables, d_tables, stream));
    else if (tables <= (size_t)kBlobLarge * 16) NA_CUDA(upload_by_value<kBlobLarge>(h.data(), tables, d_tables, stream));
    else NA_CUDA(cudaMemcpyAsync(d_tables, h.data(), tables, cudaMemcpyHostToDevice, stream));   // pageable: staged before the call returns
    RepackParams rp;
    rp.coords = (const float*)coords; rp.pk = d_pk;
    rp.off = (const int32_t*)(d_tables + o_off); rp.pad_off = (const uint32_t*)(d_tables + o_pad);
    rp.range_keys = scalars + 4; rp.reset = scalars + 16; rp.boxes = (const BoxConst*)(d_tables + o_boxes);
    rp.n_species = n_species; rp.n_total = off[n_species]; rp.n_frames = n_frames;
    rp.box_type = box_type; rp.n_boxes = nb > 0 ? nb : 1;
    rp.frame_slots = frame_slots; rp.blocks_per_frame = blocks_per_frame;
    rp.zero = nullptr; rp.zero_count = 0;
    repack_kernel<<<blocks_per_frame * (uint32_t)n_frames, 256, 0, stream>>>(rp);
    NA_CUDA(cudaGetLastError());
    if (wt.n_items == 0) return CDH_OK;
    TileParams tp;
    tp.segs = (const Seg*)d_tables; tp.rows = (const Row*)(d_tables + o_rows); tp.descs = nullptr;
    tp.counter = scalars; tp.out = (unsigned long long*)out; tp.range_keys = scalars + 4; tp.win_lo = nullptr;
    tp.n_rows = (uint32_t)wt.rows.size() - 1; tp.n_items = (uint32_t)wt.n_items; tp.n_bins = (uint32_t)n_bins; tp.tj = tj;
    tp.smem_bins = (uint32_t)n_bins; tp.n_stages = (uint32_t)n_stages;
    tp.pk = d_pk; tp.boxes = (const BoxConst*)(d_tables + o_boxes);
    tp.rmax = rmax_f; tp.scale = scale_f; tp.thr2_bits = d2_threshold_bits(rmax_f); tp.one = 1.0f; tp.one_u = 1.0f;
    tp.range_lo = -INFINITY; tp.range_hi = INFINITY; tp.keep_bins = 0u; tp.claim_ahead = 1u;
    void* args[1] = {(void*)&tp};
    const uint32_t grid = grid_full < tp.n_items ? grid_full : tp.n_items;
    NA_CUDA(cudaLaunchKernel(v.fn, dim3(grid), dim3((unsigned)v.threads), args, (size_t)smem_bytes, stream));
    return CDH_OK;
}
