// cdh_f64.cuh -- the double-precision path (precision == CDH_F64; SURVEY.md 8(f) "next" row 1; the paper's second
// template instantiation).
//
// Same steps S0-S7 and the same work tables as the fp32 path, but the per-pair arithmetic is the pinned sequence
// spelled out with the IEEE double intrinsics (__dsub_rn, __dmul_rn, __dadd_rn, __dsqrt_rn, rint, floor): there are
// no packed forms or magic-number shortcuts in double.  The one shortcut is the triclinic pruning (exact, see
// DESIGN.md "Triclinic pruning"; the margins are far wider in double).
//
// Layout: groups of 4 particles, 12 doubles per group  x0..3 | y0..3 | z0..3  (96 bytes), NaN padded like the fp32
// buffer; a j-stage is 256 particles = 6 KB, the ring of stages is filled by 1-D TMA bulk copies (cdh_sched.cuh).
#pragma once
#include "cdh_kernels.cuh"
#include "cdh_sqrt64.cuh"

namespace cdh {

constexpr int kStageBytes64 = kStageGroups * kGroupFloats * 8;

struct BoxConst64 {
    double L[3], invL[3];       // ORTHO
    double B[9], Binv[9];       // TRICLINIC, row-major, columns of B = box vectors
    double S[27][3];            // shift vectors
    double prune_ok;            // 1: the zero-shift candidate may decide alone (r_max <= h_min/2, conditioning)
    double pad_;
};

struct TileParams64 : TileCommon {
    const double*   pk;
    const BoxConst64* boxes;
    double rmax, scale;         // r_max, n_bins / r_max
    uint32_t keep_bins;         // orthorhombic full-range private histogram (as TileParams::keep_bins), else 0
    BoxConst64 box0;            // PBOX variants (one box for all frames): the constants sit in the kernel-parameter
                                // constant bank and are used as c[0x0][..] operands, no shared-memory loads
};

// ---- K0 for doubles ------------------------------------------------------------------------------
struct RepackParams64 {
    const double* coords;       // [n_frames][n_total][3]
    double* pk;
    const int32_t* off;
    const uint32_t* pad_off;
    unsigned int* range_keys;
    unsigned int* reset;        // as RepackParams
    const BoxConst64* boxes;
    int32_t n_species, n_total, n_frames;
    int32_t box_type, n_boxes;
    uint32_t frame_slots;
    uint32_t blocks_per_frame;
    unsigned long long* zero;   // as RepackParams
    uint64_t zero_count;
};

static __global__ void __launch_bounds__(256) repack_kernel_f64(const RepackParams64 P) {
    pdl_launch_dependents();
    if (blockIdx.x == 0 && threadIdx.x < 16) P.reset[threadIdx.x] = 0u;
    if (P.zero != nullptr)
        for (uint64_t k = (uint64_t)blockIdx.x * 256u + threadIdx.x; k < P.zero_count; k += (uint64_t)gridDim.x * 256u) P.zero[k] = 0ull;
    const uint32_t f = blockIdx.x / P.blocks_per_frame;
    const uint32_t slot = (blockIdx.x % P.blocks_per_frame) * blockDim.x + threadIdx.x;
    float fr[3] = {0.0f, 0.0f, 0.0f}, fr_lo[3] = {0.0f, 0.0f, 0.0f};     // upper / lower float bounds of the keyed quantity
    bool have = false;
    if (slot < P.frame_slots) {
        int lo = 0, hi = P.n_species;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(P.pad_off + mid) <= slot) lo = mid; else hi = mid;
        }
        const uint32_t k = slot - __ldg(P.pad_off + lo);
        const int32_t n = __ldg(P.off + lo + 1) - __ldg(P.off + lo);
        double x = __longlong_as_double(0x7ff8000000000000ll), y = x, z = x;   // NaN padding
        if (k < (uint32_t)n) {
            const double* c = P.coords + ((size_t)f * P.n_total + (size_t)__ldg(P.off + lo) + k) * 3;
            x = c[0]; y = c[1]; z = c[2];
            if (P.box_type == BOX_TRI) {      // only the triclinic pruning reads the range
                const BoxConst64* bc = P.boxes + (P.n_boxes == 1 ? 0 : f);
#pragma unroll
                for (int q = 0; q < 3; ++q) fr[q] = fr_lo[q] = (float)(bc->Binv[3 * q] * x + bc->Binv[3 * q + 1] * y + bc->Binv[3 * q + 2] * z);
                have = (fr[0] == fr[0]) && (fr[1] == fr[1]) && (fr[2] == fr[2]);
            } else if (P.box_type == BOX_ORTHO) {   // the full-range CLEAN form needs |x / L| < 2^20 (cdh_math: launch_begin)
                const BoxConst64* bc = P.boxes + (P.n_boxes == 1 ? 0 : f);
                fr[0] = fr_lo[0] = (float)(x * bc->invL[0]); fr[1] = fr_lo[1] = (float)(y * bc->invL[1]); fr[2] = fr_lo[2] = (float)(z * bc->invL[2]);
                have = (fr[0] == fr[0]) && (fr[1] == fr[1]) && (fr[2] == fr[2]);
            } else {                                // no box: float bounds of the coordinates, rounded OUTWARD
                fr[0] = __double2float_ru(x); fr[1] = __double2float_ru(y); fr[2] = __double2float_ru(z);
                fr_lo[0] = __double2float_rd(x); fr_lo[1] = __double2float_rd(y); fr_lo[2] = __double2float_rd(z);
                have = (x == x) && (y == y) && (z == z);
            }
            if (!((x == x) && (y == y) && (z == z))) atomicOr(P.range_keys + 6, 1u);
        }
        double* g = P.pk + ((size_t)f * (P.frame_slots / kGroup) + slot / kGroup) * kGroupFloats + (slot % kGroup);
        g[0] = x; g[4] = y; g[8] = z;
    }
    {
        __shared__ unsigned int s_keys[6];
        if (threadIdx.x < 6) s_keys[threadIdx.x] = 0u;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            uint32_t kmax = have ? float_key(fr[q]) : 0u, kmin_c = have ? ~float_key(fr_lo[q]) : 0u;
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

// No box: an UPPER bound of every pinned d2 of the call in double, from the outward-rounded float bounds of the coordinates
// (cf. coord_extent2_ru); +inf when a coordinate is NaN.
__device__ __forceinline__ double coord_extent2_ru64(const unsigned int* __restrict__ keys) {
    if (__ldg(keys + 6) != 0u) return __longlong_as_double(0x7ff0000000000000ll);
    double acc = 0.0;
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const uint32_t kmax = __ldg(keys + q), kmin_c = __ldg(keys + 3 + q);
        if (kmax != 0u) {
            const double ext = __dsub_ru((double)key_float(kmax), (double)key_float(~kmin_c));
            acc = __dadd_ru(acc, __dmul_ru(ext, ext));
        }
    }
    return acc;
}

// ---- the pinned sequence in double ---------------------------------------------------------------
constexpr double kPruneLimit64 = 0.5 - 9.313225746154785e-10;     // 1/2 - 2^-30
constexpr float kPruneRange64 = 1024.0f;                          // fractional range up to which pruning is proven

// d2 of one pair.  prune: the zero-shift candidate may be accepted when every |s_k - n_k| <= 1/2 - 2^-30.
struct OrthoRegs64 { double L[3], invL[3]; };      // the orthorhombic constants, held in registers

template <int BOX>
__device__ __forceinline__ double pair_d2_f64(double xi, double yi, double zi, double xj, double yj, double zj,
                                              const BoxConst64& bcr, const OrthoRegs64& ob, bool prune) {
    const BoxConst64* __restrict__ bc = &bcr;
    double dx = __dsub_rn(xj, xi), dy = __dsub_rn(yj, yi), dz = __dsub_rn(zj, zi);
    if constexpr (BOX == BOX_ORTHO) {
        double n;
        n = rint(__dmul_rn(dx, ob.invL[0])); dx = __dsub_rn(dx, __dmul_rn(ob.L[0], n));
        n = rint(__dmul_rn(dy, ob.invL[1])); dy = __dsub_rn(dy, __dmul_rn(ob.L[1], n));
        n = rint(__dmul_rn(dz, ob.invL[2])); dz = __dsub_rn(dz, __dmul_rn(ob.L[2], n));
    } else if constexpr (BOX == BOX_TRI) {
        double n[3], e[3], fm = 0.0;
        const double d[3] = {dx, dy, dz};
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double s = __dadd_rn(__dadd_rn(__dmul_rn(bc->Binv[3 * k + 0], dx), __dmul_rn(bc->Binv[3 * k + 1], dy)),
                                       __dmul_rn(bc->Binv[3 * k + 2], dz));
            n[k] = rint(s);
            fm = fmax(fm, fabs(__dsub_rn(s, n[k])));      // NaN: ignored (the pair is dropped either way)
        }
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            const double sh = __dadd_rn(__dadd_rn(__dmul_rn(bc->B[3 * r + 0], n[0]), __dmul_rn(bc->B[3 * r + 1], n[1])),
                                        __dmul_rn(bc->B[3 * r + 2], n[2]));
            e[r] = __dsub_rn(d[r], sh);
        }
        if (prune && fm <= kPruneLimit64)
            return __dadd_rn(__dadd_rn(__dmul_rn(e[0], e[0]), __dmul_rn(e[1], e[1])), __dmul_rn(e[2], e[2]));
        double best = __longlong_as_double(0x7ff0000000000000ll);
#pragma unroll 1
        for (int m = 0; m < 27; ++m) {
            const double cx = __dadd_rn(e[0], bc->S[m][0]), cy = __dadd_rn(e[1], bc->S[m][1]), cz = __dadd_rn(e[2], bc->S[m][2]);
            const double c2 = __dadd_rn(__dadd_rn(__dmul_rn(cx, cx), __dmul_rn(cy, cy)), __dmul_rn(cz, cz));
            if (c2 < best) best = c2;
        }
        return best;
    }
    return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// CLEAN (cdh_sched.cuh KIND_CLEAN, MODE_SHARED): the caller promises that every pair of the stage may be binned where it
// falls -- no box: d < r_max for every pair (the flushed slots end with the Q3 clamp as usual); orthorhombic full-range
// histogram: dropped pairs land in slots beyond the flushed ones -- so the DSETP compare and the select are left out.
template <int MODE, bool CLEAN, bool CLAMP>
__device__ __forceinline__ void bin_f64(double d2, double rmax, double scale, const HistView& hv, bool keep) {
    const double d = sqrt_rn_f64(d2);
    const uint32_t f = __double2uint_rd(__dmul_rn(d, scale));   // floor, saturating (one F2I)
    if constexpr (CLEAN && MODE == MODE_SHARED) {
        hist_inc(hv.hist_addr + 4u * (CLAMP ? min(f, hv.last_bin) : f));
        return;
    }
    const uint32_t bin = min(f, hv.last_bin);                   // reading Q3
    const uint32_t b = bin - hv.lo;                             // unsigned wrap for bins below the sweep / window
    bool ok = keep && (d < rmax);                               // false for NaN (NaN input, +inf)
    if constexpr (MODE == MODE_GLOBAL) { red_global_inc_if(ok, hv.grow + bin); return; }
    if constexpr (MODE == MODE_HYBRID) {
        const bool in = ok && b < hv.lim;
        hist_inc(in ? hv.hist_addr + 4u * b : hv.trash_addr);
        red_global_inc_if(ok && !in, hv.grow + bin);
        return;
    }
    if constexpr (MODE == MODE_SPLIT) ok = ok && b < hv.lim;
    hist_inc(ok ? hv.hist_addr + 4u * b : hv.trash_addr);
}

// ---- the arithmetic policy of the double-precision tile kernel (cdh_sched.cuh) -----------------------
template <int BOX, bool PBOX>
struct MathF64 {
    using Real = double;
    using Box = BoxConst64;
    using Params = TileParams64;
    static constexpr int kStageBytes = kStageBytes64;
    static constexpr bool kPeriodic = BOX != BOX_NONE;
    static constexpr bool kHasClean = BOX == BOX_NONE || BOX == BOX_ORTHO;
    static constexpr bool kCleanPadded = false;
    static constexpr int kUnroll = 1;
    struct Launch { bool range_ok; bool clean; };
    struct Item {
        double xi[4], yi[4], zi[4];
        OrthoRegs64 ob;
        bool prune;
    };

    __device__ __forceinline__ static bool launch_begin(const Params& P, Launch& L) {
        L.clean = false;
        L.range_ok = (BOX == BOX_TRI) ? (frac_range(P.range_keys) <= kPruneRange64) : true;
        // no box: every pinned d is below r_max (sqrt is monotone and correctly rounded) and no coordinate is NaN
        if constexpr (BOX == BOX_NONE) L.clean = __dsqrt_rn(coord_extent2_ru64(P.range_keys)) < P.rmax;
        // orthorhombic: the host sized the private histogram for half the box diagonal; the wrapped components stay within
        // L/2 (1 + 2^-20) while |x / L| < 2^20 (the double product is then exact to 2^-32); no NaN coordinate
        if constexpr (BOX == BOX_ORTHO) L.clean = P.keep_bins != 0u && __ldg(P.range_keys + 6) == 0u && frac_range(P.range_keys) <= 1048576.0f;
        return true;
    }
    template <int MODE>
    __device__ __forceinline__ static void key_begin(const Params& P, const Launch&, const Seg& seg, HistView& hv) {
        if constexpr (MODE == MODE_HYBRID) {
            hv.lo = min(__ldg(P.win_lo + seg.hist), P.n_bins - min(P.n_bins, P.smem_bins));
            hv.lim = min(P.smem_bins, P.n_bins - hv.lo);
        } else {
            hv.lo = seg.bin_lo; hv.lim = seg.bin_cnt + seg.last_sweep;
            if constexpr (BOX == BOX_ORTHO && MODE == MODE_SHARED) if (P.keep_bins != 0u) hv.lim = P.keep_bins;
        }
    }
    __device__ __forceinline__ static void item_begin(const Params&, const Launch& L, const double* __restrict__ g, const Box* s_box,
                                                      const HistView&, Item& it) {
        const double2* gi = reinterpret_cast<const double2*>(g);      // one group of 12 doubles
        { const double2 a = __ldg(gi), b = __ldg(gi + 1); it.xi[0] = a.x; it.xi[1] = a.y; it.xi[2] = b.x; it.xi[3] = b.y; }
        { const double2 a = __ldg(gi + 2), b = __ldg(gi + 3); it.yi[0] = a.x; it.yi[1] = a.y; it.yi[2] = b.x; it.yi[3] = b.y; }
        { const double2 a = __ldg(gi + 4), b = __ldg(gi + 5); it.zi[0] = a.x; it.zi[1] = a.y; it.zi[2] = b.x; it.zi[3] = b.y; }
        it.prune = (BOX == BOX_TRI) ? (L.range_ok && s_box->prune_ok != 0.0) : true;
        if constexpr (BOX == BOX_ORTHO) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { it.ob.L[k] = s_box->L[k]; it.ob.invL[k] = s_box->invL[k]; }
        }
    }
    template <int MODE, int KIND, bool SKIPV = false>
    __device__ __forceinline__ static void group(const Params& P, const Launch&, const Item& it, const unsigned char* stage,
                                                 uint32_t g, uint32_t jg, uint32_t ig, const HistView& hv, const Box* s_box) {
        constexpr bool MASKED = KIND == KIND_MASKED;
        const double2* sj = reinterpret_cast<const double2*>(stage);
#pragma unroll
        for (int h = 0; h < 2; ++h) {                   // two j-particles at a time (register pressure)
            const double2 XJ = sj[6 * g + h], YJ = sj[6 * g + 2 + h], ZJ = sj[6 * g + 4 + h];
            const double xj[2] = {XJ.x, XJ.y}, yj[2] = {YJ.x, YJ.y}, zj[2] = {ZJ.x, ZJ.y};
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int r = 0; r < kR; ++r) {
                    const bool keep = !MASKED || (jg + 2 * h + c > ig + r);
                    double d2;
                    if constexpr (PBOX) d2 = pair_d2_f64<BOX>(it.xi[r], it.yi[r], it.zi[r], xj[c], yj[c], zj[c], P.box0, it.ob, it.prune);
                    else d2 = pair_d2_f64<BOX>(it.xi[r], it.yi[r], it.zi[r], xj[c], yj[c], zj[c], *s_box, it.ob, it.prune);
                    bin_f64<MODE, KIND == KIND_CLEAN, BOX == BOX_NONE>(d2, P.rmax, P.scale, hv, keep);
                }
        }
    }
};

}  // namespace cdh
