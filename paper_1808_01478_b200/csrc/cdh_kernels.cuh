// cdh_kernels.cuh -- the CUDA kernels of libcdh (sm_100a).
//
//   K0 repack_kernel      S0: AoS xyz -> padded groups of 4 (cdh_device.cuh), coordinate extent
//   K1 tile_kernel<...>   S1 tile schedule, S2 distance, S3 minimum image, S4 bin, S5 private
//                         shared-memory histogram, S6/S7 flush into the uint64 result
// (step names: SURVEY.md 8a; the paper's analogue is the shared-memory kernel).
//
// The per-pair arithmetic reproduces DESIGN.md "Pinned sequence" bit for bit.  VAR_SIMPLE spells it
// with the CUDA library's IEEE intrinsics (__fsub_rn, __fmul_rn, __fadd_rn, __fsqrt_rn, rintf, floorf);
// VAR_FAST computes the same integers with packed f32x2 arithmetic, a magic-number rint/floor, a
// Newton-corrected MUFU.RSQ square root and a threshold on d2.
#pragma once
#include "cdh_sched.cuh"

namespace cdh {

constexpr int VAR_SIMPLE = 0;
constexpr int VAR_FAST = 1;
// Two more forms of the plain kernel's histogram update, for measuring what the hardware merge of equal addresses in
// ATOMS.POPC.INC is worth: software aggregation of equal bins with __match_any_sync
// and one ATOMS.ADD per distinct bin (CDH_FLAG_WARP_AGGREGATE), and one ATOMS.ADD per lane (CDH_FLAG_NO_AGGREGATE).
constexpr int VAR_SIMPLE_MATCH = 2;
constexpr int VAR_SIMPLE_PLAIN = 3;

constexpr int BOX_NONE = 0, BOX_ORTHO = 1, BOX_TRI = 2;

// Triclinic zero structure (skipping a term whose matrix entry is exactly 0 in B and in B^-1 changes
// at most the sign of a zero, never d2): 0 general 3x3, 1 upper triangular (a along x, b in the xy
// plane), 2 upper triangular with B[0][1] == 0 as well (the rhombic dodecahedron of config 3).
constexpr int TRI_GENERAL = 0, TRI_UPPER = 1, TRI_UPPER_B01 = 2;
// + TRI_WIDE: coordinates spanning up to 64 cells (unwrapped trajectories): n_k is no longer in {-1,0,1}, so B*n uses the
// pinned multiply / add chain and the pruning margin grows with the measured range (cdh_tile.cuh).
constexpr int TRI_WIDE = 4;
// For BOX_ORTHO the same template slot selects the rint form (cdh_fast.cuh): 0 the pinned 5-operation form, 1 fused
// (3 operations per axis; needs the host-searched constants), 2 exact-product form (4 operations; n in {-1,0,1}).
constexpr int ORTHO_PLAIN = 0, ORTHO_FUSED = 1, ORTHO_EXACT = 2;

// ---------------------------------------------------------------------------------------------
// K0: repack.  One thread per padded particle slot of one frame.
// ---------------------------------------------------------------------------------------------
struct RepackParams {
    const float* coords;        // [n_frames][n_total][3]
    float* pk;                  // [n_frames][frame_groups][12]
    const int32_t* off;         // device, [n_species+1] particle offsets
    const uint32_t* pad_off;    // device, [n_species+1] padded particle offsets (multiples of kPadParticles)
    unsigned int* range_keys;   // device, [7]: atomicMax of key(f_k) (k = 0..2) and of ~key(f_k) (3..5), f = b^-1 x
                                // (fractional coordinates, approximate; the raw coordinates when there is no box), [6] is set
                                // when a particle has a NaN coordinate; zero-initialised; see frac_range() / coord_extent2_ru()
    unsigned int* reset;        // the 16 scalars of the context's NEXT call, zeroed here (cdh_api.cu "d_scalars")
    const BoxConst* boxes;      // box constants (periodic boxes), one or n_frames
    int32_t n_species, n_total, n_frames;
    int32_t box_type, n_boxes;
    uint32_t frame_slots;       // padded particles per frame
    uint32_t blocks_per_frame;
    unsigned long long* zero;   // the call's result, zeroed here (grid-stride) unless the call accumulates: nullptr then
    uint64_t zero_count;        // uint64 elements of it
};

// Order-preserving map float -> uint32 (never 0 for a non-NaN float except -NaN patterns, which are excluded).
__device__ __forceinline__ uint32_t float_key(float v) {
    const uint32_t b = __float_as_uint(v);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key_float(uint32_t k) {
    return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
// Largest extent over the three axes of the fractional coordinates of all particles of the call (0 if none), made
// conservative for coordinates far from the origin: the keys come from fp32 evaluations of b^-1 x whose absolute
// error grows with |b^-1 x|, so the result is max(max - min, max|b^-1 x| * 1.49 / 4096): the 1.49 limit of the fused
// rint / exact-B*n paths then also implies |b^-1 x| <= 4096 (range error < 1e-3, far inside the 0.01 margin to 3/2),
// and the 2^20 limit of the magic-number rint implies |b^-1 x| < 2^32.
__device__ __forceinline__ float frac_range(const unsigned int* __restrict__ keys) {
    float r = 0.0f;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const uint32_t kmax = __ldg(keys + q), kmin_c = __ldg(keys + 3 + q);
        if (kmax != 0u) {
            const float hi = key_float(kmax), lo = key_float(~kmin_c);
            r = fmaxf(r, fmaxf(hi - lo, fmaxf(fabsf(hi), fabsf(lo)) * (1.49f / 4096.0f)));
        }
    }
    return r;
}

// No box: an UPPER bound of every pinned d2 of the call, sum over the axes of (max - min)^2 with every operation rounded
// up (subtraction, square and sum are monotone, so the round-to-nearest d2 of any pair is below it).  +inf when a
// particle has a NaN coordinate; 0 when there are no particles.
__device__ __forceinline__ float coord_extent2_ru(const unsigned int* __restrict__ keys) {
    if (__ldg(keys + 6) != 0u) return __int_as_float(0x7f800000);
    float acc = 0.0f;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const uint32_t kmax = __ldg(keys + q), kmin_c = __ldg(keys + 3 + q);
        if (kmax != 0u) {
            const float ext = __fsub_ru(key_float(kmax), key_float(~kmin_c));
            acc = __fadd_ru(acc, __fmul_ru(ext, ext));
        }
    }
    return acc;
}

static __global__ void __launch_bounds__(256) repack_kernel(const RepackParams P) {
    pdl_launch_dependents();    // the tile kernel may start its prologue; it waits for this grid to complete before it reads pk
    if (blockIdx.x == 0 && threadIdx.x < 16) P.reset[threadIdx.x] = 0u;
    if (P.zero != nullptr)      // saves the call one memset node (small calls are launch-latency bound)
        for (uint64_t k = (uint64_t)blockIdx.x * 256u + threadIdx.x; k < P.zero_count; k += (uint64_t)gridDim.x * 256u) P.zero[k] = 0ull;
    const uint32_t f = blockIdx.x / P.blocks_per_frame;
    const uint32_t slot = (blockIdx.x % P.blocks_per_frame) * blockDim.x + threadIdx.x;
    float fr[3] = {0.0f, 0.0f, 0.0f};
    bool have = false;
    if (slot < P.frame_slots) {
        // species of this slot: largest s with pad_off[s] <= slot
        int lo = 0, hi = P.n_species;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(P.pad_off + mid) <= slot) lo = mid; else hi = mid;
        }
        const uint32_t k = slot - __ldg(P.pad_off + lo);
        const int32_t n = __ldg(P.off + lo + 1) - __ldg(P.off + lo);
        float x = __int_as_float(0x7fc00000), y = x, z = x;   // NaN padding
        if (k < (uint32_t)n) {
            const float* c = P.coords + ((size_t)f * P.n_total + (size_t)__ldg(P.off + lo) + k) * 3;
            x = c[0]; y = c[1]; z = c[2];
            // Fractional coordinates b^-1 x (approximate: only their range is compared against limits with wide
            // margins).  A particle with a NaN coordinate is left out: its pairs are dropped anyway.
            if (P.box_type == BOX_ORTHO) {
                const BoxConst* bc = P.boxes + (P.n_boxes == 1 ? 0 : f);
                fr[0] = x * bc->invL[0]; fr[1] = y * bc->invL[1]; fr[2] = z * bc->invL[2];
                have = true;
            } else if (P.box_type == BOX_TRI) {
                const BoxConst* bc = P.boxes + (P.n_boxes == 1 ? 0 : f);
#pragma unroll
                for (int q = 0; q < 3; ++q) fr[q] = bc->Binv[3 * q] * x + bc->Binv[3 * q + 1] * y + bc->Binv[3 * q + 2] * z;
                have = true;
            } else {
                fr[0] = x; fr[1] = y; fr[2] = z;            // no box: the extent of the coordinates themselves
                have = true;
            }
            have = have && (fr[0] == fr[0]) && (fr[1] == fr[1]) && (fr[2] == fr[2]);
            if (!((x == x) && (y == y) && (z == z))) atomicOr(P.range_keys + 6, 1u);   // rare: a NaN input coordinate
        }
        float* g = P.pk + ((size_t)f * (P.frame_slots / kGroup) + slot / kGroup) * kGroupFloats + (slot % kGroup);
        g[0] = x; g[4] = y; g[8] = z;
    }
    {
        // CTA max / min of the order-preserving keys (shared atomics), then one global atomic per key and CTA
        __shared__ unsigned int s_keys[6];
        if (threadIdx.x < 6) s_keys[threadIdx.x] = 0u;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            uint32_t kmax = have ? float_key(fr[q]) : 0u, kmin_c = have ? ~float_key(fr[q]) : 0u;
            for (int o = 16; o > 0; o >>= 1) {
                kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
                kmin_c = max(kmin_c, __shfl_xor_sync(0xffffffffu, kmin_c, o));
            }
            if ((threadIdx.x & 31) == 0 && kmax != 0u) { atomicMax(&s_keys[q], kmax); atomicMax(&s_keys[3 + q], kmin_c); }
        }
        __syncthreads();
        if (threadIdx.x < 6 && s_keys[threadIdx.x] != 0u) atomicMax(P.range_keys + threadIdx.x, s_keys[threadIdx.x]);
    }
}

// ---------------------------------------------------------------------------------------------
// K0b: window_kernel (MODE_HYBRID, very wide histograms).  One CTA per histogram row samples pairs of the row's first
// segment, bins their APPROXIMATE distances (plain float arithmetic, Eq. 5 without the neighbour search) into 1024
// coarse cells and writes the first bin of the `window` consecutive bins that hold the most samples: the tile kernel
// keeps that window of the row in shared memory and sends the rest to L2.  The choice only affects speed, never the
// result, so nothing here belongs to the pinned sequence.
// ---------------------------------------------------------------------------------------------
constexpr int kWindowCells = 1024;
constexpr int kWindowSamplesPerThread = 64;

template <class Real, class Box>
struct WindowParams {
    const Real* pk;
    const Seg* segs;
    const int32_t* row_seg;     // [n_hist] first segment of each histogram row, -1 if the row has no pairs
    const Box* boxes;
    uint32_t* win_lo;           // [n_hist] out
    int32_t box_type;
    uint32_t n_bins, window;    // window: bins the shared histogram holds
    float scale;                // n_bins / r_max
};

__device__ __forceinline__ uint32_t window_hash(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

template <class Real, class Box>
__global__ void __launch_bounds__(256) window_kernel(const WindowParams<Real, Box> P) {
    __shared__ uint32_t cells[kWindowCells];
    __shared__ uint32_t best_lo;
    for (int k = threadIdx.x; k < kWindowCells; k += 256) cells[k] = 0;
    __syncthreads();
    const int32_t sid = __ldg(P.row_seg + blockIdx.x);
    if (sid < 0) { if (threadIdx.x == 0) P.win_lo[blockIdx.x] = 0; return; }
    const Seg seg = P.segs[sid];
    const Box* bc = P.boxes + seg.box;
    auto coord = [&](uint32_t group0, uint32_t k, float (&x)[3]) {
        const Real* g = P.pk + ((size_t)group0 + (k >> 2)) * kGroupFloats + (k & 3u);
        x[0] = (float)g[0]; x[1] = (float)g[4]; x[2] = (float)g[8];
    };
    for (int s = 0; s < kWindowSamplesPerThread; ++s) {
        const uint32_t h = window_hash((blockIdx.x * 256u + threadIdx.x) * kWindowSamplesPerThread + s + 0x9e3779b9u);
        const uint32_t i = __umulhi(h, (uint32_t)seg.ni), j = __umulhi(window_hash(h ^ 0x85ebca6bu), (uint32_t)seg.nj);
        float a[3], b[3], d[3];
        coord(seg.i_group, i, a); coord(seg.j_group, j, b);
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] = b[c] - a[c];
        if (P.box_type == BOX_ORTHO) {
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] -= (float)bc->L[c] * rintf(d[c] * (float)bc->invL[c]);
        } else if (P.box_type == BOX_TRI) {
            float n[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) n[k] = rintf((float)bc->Binv[3 * k] * d[0] + (float)bc->Binv[3 * k + 1] * d[1] + (float)bc->Binv[3 * k + 2] * d[2]);
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] -= (float)bc->B[3 * c] * n[0] + (float)bc->B[3 * c + 1] * n[1] + (float)bc->B[3 * c + 2] * n[2];
        }
        const float t = sqrtf(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]) * P.scale;      // NaN / out of range: not counted
        if (t >= 0.0f && t < (float)P.n_bins)
            atomicAdd(&cells[min((uint32_t)(t * ((float)kWindowCells / (float)P.n_bins)), (uint32_t)kWindowCells - 1u)], 1u);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        // sliding window of w cells over the coarse histogram; the first maximum wins
        const uint32_t w = max(1u, (uint32_t)(((uint64_t)P.window * kWindowCells) / P.n_bins));
        uint32_t sum = 0, best = 0, lo = 0;
        for (uint32_t c = 0; c < (uint32_t)kWindowCells; ++c) {
            sum += cells[c];
            if (c >= w) sum -= cells[c - w];
            if (sum > best) { best = sum; lo = c + 1 >= w ? c + 1 - w : 0; }
        }
        best_lo = (uint32_t)(((uint64_t)lo * P.n_bins) / kWindowCells);
        P.win_lo[blockIdx.x] = min(best_lo, P.n_bins - min(P.n_bins, P.window));
    }
}

// ---------------------------------------------------------------------------------------------
// Box constants staged in shared memory (triclinic) / registers (orthorhombic)
// ---------------------------------------------------------------------------------------------
struct OrthoRegs { float L[3], invL[3]; };

// The pinned sequence for ONE pair, spelled with IEEE intrinsics.  Returns d2.
// bc: box constants (global or shared memory pointer); only read for periodic boxes.
template <int BOX>
__device__ __forceinline__ float pair_d2_simple(float xi, float yi, float zi, float xj, float yj, float zj,
                                                const BoxConst* __restrict__ bc) {
    float dx = __fsub_rn(xj, xi), dy = __fsub_rn(yj, yi), dz = __fsub_rn(zj, zi);
    if constexpr (BOX == BOX_ORTHO) {
        float t, n;
        t = __fmul_rn(dx, bc->invL[0]); n = rintf(t); dx = __fsub_rn(dx, __fmul_rn(bc->L[0], n));
        t = __fmul_rn(dy, bc->invL[1]); n = rintf(t); dy = __fsub_rn(dy, __fmul_rn(bc->L[1], n));
        t = __fmul_rn(dz, bc->invL[2]); n = rintf(t); dz = __fsub_rn(dz, __fmul_rn(bc->L[2], n));
    } else if constexpr (BOX == BOX_TRI) {
        float n[3], e[3];
        const float d[3] = {dx, dy, dz};
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float s = __fadd_rn(__fadd_rn(__fmul_rn(bc->Binv[3 * k + 0], dx), __fmul_rn(bc->Binv[3 * k + 1], dy)),
                                      __fmul_rn(bc->Binv[3 * k + 2], dz));
            n[k] = rintf(s);
        }
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            const float sh = __fadd_rn(__fadd_rn(__fmul_rn(bc->B[3 * r + 0], n[0]), __fmul_rn(bc->B[3 * r + 1], n[1])),
                                       __fmul_rn(bc->B[3 * r + 2], n[2]));
            e[r] = __fsub_rn(d[r], sh);
        }
        float best = __int_as_float(0x7f800000);
#pragma unroll 1
        for (int m = 0; m < 27; ++m) {
            const float cx = __fadd_rn(e[0], bc->S[m][0]), cy = __fadd_rn(e[1], bc->S[m][1]),
                        cz = __fadd_rn(e[2], bc->S[m][2]);
            const float c2 = __fadd_rn(__fadd_rn(__fmul_rn(cx, cx), __fmul_rn(cy, cy)), __fmul_rn(cz, cz));
            if (c2 < best) best = c2;
        }
        return best;
    }
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// Binning of one d2 by the pinned sequence (library sqrt / floor).  hist = shared address of slot 0,
// the CTA owns bins [bin_lo, bin_lo + lim).  Must be called by all 32 lanes of the warp (keep = false for a pair
// that does not exist): the VAR_SIMPLE_MATCH form synchronises the warp.
template <int VAR, int MODE>
__device__ __forceinline__ void bin_simple(float d2, bool keep, float rmax, float scale, uint32_t n_bins,
                                           uint32_t hist, uint32_t bin_lo, uint32_t lim, unsigned long long* __restrict__ grow) {
    const float d = __fsqrt_rn(d2);
    keep = keep && (d < rmax);                            // drops d >= r_max and NaN
    uint32_t b = 0xFFFFFFFFu;
    if (keep) {
        b = (uint32_t)fminf(floorf(__fmul_rn(d, scale)), 4294967040.0f);
        b = min(b, n_bins - 1u) - bin_lo;                 // reading Q3; unsigned wrap for bins below the sweep
        if (!(b < lim)) b = 0xFFFFFFFFu;
    }
    if constexpr (MODE == MODE_GLOBAL) {
        if (b != 0xFFFFFFFFu) atomicAdd(grow + b, 1ull);      // bin_lo = 0, lim = n_bins + 1 in this mode
    } else if constexpr (VAR == VAR_SIMPLE_MATCH) {
        const uint32_t peers = __match_any_sync(0xffffffffu, b);
        if (b != 0xFFFFFFFFu && (uint32_t)(__ffs(peers) - 1) == (threadIdx.x & 31u)) hist_add(hist + 4u * b, (uint32_t)__popc(peers));
    } else if constexpr (VAR == VAR_SIMPLE_PLAIN) {
        if (b != 0xFFFFFFFFu) hist_add(hist + 4u * b, 1u + (n_bins >> 31));     // a register operand: ATOMS.ADD, not POPC.INC
    } else {
        if (b != 0xFFFFFFFFu) hist_inc(hist + 4u * b);
    }
}

}  // namespace cdh
