// cdh_f64.cuh -- the double-precision path (precision == CDH_F64; SURVEY.md 8(f) "next" row 1; the paper's second
// template instantiation).
//
// Same steps S0-S7 and the same work tables as the fp32 path, but the per-pair arithmetic is the pinned sequence
// spelled out with the IEEE double intrinsics (__dsub_rn, __dmul_rn, __dadd_rn, __dsqrt_rn, rint, floor): there are
// no packed forms or magic-number shortcuts in double.  The one shortcut is the triclinic pruning (exact, see
// DESIGN.md "Triclinic pruning"; the margins are far wider in double).
//
// Layout: groups of 4 particles, 12 doubles per group  x0..3 | y0..3 | z0..3  (96 bytes), NaN padded like the fp32
// buffer; a j-stage is 256 particles = 6 KB, two stages filled by 1-D TMA bulk copies.
#pragma once
#include "cdh_tile.cuh"
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

struct TileParams64 {
    const double*   pk;
    const Seg*      segs;
    const Row*      rows;
    const BoxConst64* boxes;
    unsigned int*   counter;
    unsigned long long* out;
    const unsigned int* range_keys;
    uint32_t n_rows, n_items;
    uint32_t n_bins;
    uint32_t tj;
    uint32_t smem_bins;
    double rmax, scale;         // r_max, n_bins / r_max
    BoxConst64 box0;            // PBOX variants (one box for all frames): the constants sit in the kernel-parameter
                                // constant bank and are used as c[0x0][..] operands, no shared-memory loads
};

__host__ __device__ constexpr int tile_smem_bytes64(int smem_bins) {
    return kSmemHeader + 2 * kStageBytes64 + (int)sizeof(BoxConst64) + 16 + 4 * (smem_bins + 2);
}

// ---- K0 for doubles ------------------------------------------------------------------------------
struct RepackParams64 {
    const double* coords;       // [n_frames][n_total][3]
    double* pk;
    const int32_t* off;
    const uint32_t* pad_off;
    unsigned int* range_keys;
    const BoxConst64* boxes;
    int32_t n_species, n_total, n_frames;
    int32_t box_type, n_boxes;
    uint32_t frame_slots;
    uint32_t blocks_per_frame;
};

__global__ void __launch_bounds__(256) repack_kernel_f64(const RepackParams64 P) {
    const uint32_t f = blockIdx.x / P.blocks_per_frame;
    const uint32_t slot = (blockIdx.x % P.blocks_per_frame) * blockDim.x + threadIdx.x;
    float fr[3] = {0.0f, 0.0f, 0.0f};
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
                for (int q = 0; q < 3; ++q) fr[q] = (float)(bc->Binv[3 * q] * x + bc->Binv[3 * q + 1] * y + bc->Binv[3 * q + 2] * z);
                have = (fr[0] == fr[0]) && (fr[1] == fr[1]) && (fr[2] == fr[2]);
            }
        }
        double* g = P.pk + ((size_t)f * (P.frame_slots / kGroup) + slot / kGroup) * kGroupFloats + (slot % kGroup);
        g[0] = x; g[4] = y; g[8] = z;
    }
    if (P.box_type == BOX_TRI) {
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

template <int MODE>
__device__ __forceinline__ void bin_f64(double d2, double rmax, double scale, uint32_t last_bin, uint32_t hist,
                                        uint32_t bin_lo, uint32_t lim, uint32_t trash, bool keep,
                                        unsigned long long* __restrict__ grow) {
    const double d = sqrt_rn_f64(d2);
    const uint32_t f = __double2uint_rd(__dmul_rn(d, scale));   // floor, saturating (one F2I)
    const uint32_t b = min(f, last_bin) - bin_lo;               // reading Q3; unsigned wrap for bins below the sweep
    bool ok = keep && (d < rmax);                               // false for NaN (NaN input, +inf)
    if constexpr (MODE == MODE_GLOBAL) { if (ok) atomicAdd(grow + b, 1ull); return; }    // bin_lo = 0 in this mode
    if constexpr (MODE == MODE_SPLIT) ok = ok && b < lim;
    hist_inc(ok ? hist + 4u * b : trash);
}

// ---- K1 for doubles: same schedule, stages and flush rule as tile_kernel (cdh_tile.cuh) ------------
template <int BOX, int T, int MINB, bool PBOX, int MODE, bool SKIP = false>     // SKIP: as in cdh_tile.cuh
__global__ void __launch_bounds__(T, MINB) tile_kernel_f64(const TileParams64 P) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int TI = T * kR;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    volatile uint32_t* s_item = reinterpret_cast<volatile uint32_t*>(smem + 16);
    double* stage0 = reinterpret_cast<double*>(smem + kSmemHeader);
    BoxConst64* s_box = reinterpret_cast<BoxConst64*>(smem + kSmemHeader + 2 * kStageBytes64);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + kSmemHeader + 2 * kStageBytes64 + sizeof(BoxConst64) + 16);
    const uint32_t hist_addr = smem_u32(s_hist);
    const uint32_t bar_addr = smem_u32(bars);
    const uint32_t stage_addr = smem_u32(stage0);
    const int tid = threadIdx.x;

    if (tid == 0) { mbar_init(bar_addr, 1); mbar_init(bar_addr + 8, 1); fence_mbar_init(); }
    for (uint32_t b = tid; b <= P.smem_bins + 1; b += T) s_hist[b] = 0;
    const uint32_t trash_addr = hist_addr + 4u * (P.smem_bins + 1u);
    const bool range_ok = (BOX == BOX_TRI) ? (frac_range(P.range_keys) <= kPruneRange64) : true;
    __syncthreads();

    uint32_t stage_cnt = 0;
    uint32_t cur_key = 0xFFFFFFFFu, cur_hist = 0, cur_lo = 0, cur_lim = 0, cur_box = 0xFFFFFFFFu;
    uint64_t increments = 0;

    auto flush = [&]() {
        __syncthreads();
        if (MODE != MODE_GLOBAL && cur_key != 0xFFFFFFFFu) {
            unsigned long long* o = P.out + (size_t)cur_hist * P.n_bins;
            for (uint32_t b = tid; b < cur_lim; b += T) {
                const uint32_t v = s_hist[b];
                if (v) { s_hist[b] = 0; atomicAdd(o + min(cur_lo + b, P.n_bins - 1u), (unsigned long long)v); }
            }
        }
        increments = 0;
        __syncthreads();
    };

    for (;;) {
        if (tid == 0) *s_item = atomicAdd(P.counter, 1u);
        __syncthreads();
        const uint32_t item = *s_item;
        if (item >= P.n_items) break;
        uint32_t lo = 0, hi = P.n_rows;
        while (hi - lo > 1) {
            const uint32_t mid = (lo + hi) >> 1;
            if (__ldg(&P.rows[mid].item_prefix) <= item) lo = mid; else hi = mid;
        }
        const Row row = P.rows[lo];
        const Seg seg = P.segs[row.seg];
        const uint32_t jc = row.jc0 + (item - row.item_prefix);
        const uint32_t j0 = jc * P.tj;
        const uint32_t j1 = min((uint32_t)seg.nj, j0 + P.tj);
        const uint32_t i0 = row.i0;

        if (seg.key != cur_key || increments + (uint64_t)TI * P.tj > kMaxIncrements) {
            flush();
            cur_key = seg.key; cur_hist = seg.hist; cur_lo = seg.bin_lo;
            cur_lim = seg.bin_cnt + seg.last_sweep;
        }
        increments += (uint64_t)TI * P.tj;
        if (BOX != BOX_NONE && seg.box != cur_box) {
            __syncthreads();
            const double* src = reinterpret_cast<const double*>(P.boxes + seg.box);
            for (int k = tid; k < (int)(sizeof(BoxConst64) / 8); k += T) reinterpret_cast<double*>(s_box)[k] = __ldg(src + k);
            cur_box = seg.box;
            __syncthreads();
        }

        // my R = 4 i-particles: one group of 12 doubles
        const double2* gi = reinterpret_cast<const double2*>(P.pk + ((size_t)seg.i_group + (i0 >> 2) + tid) * kGroupFloats);
        double xi[4], yi[4], zi[4];
        { const double2 a = __ldg(gi), b = __ldg(gi + 1); xi[0] = a.x; xi[1] = a.y; xi[2] = b.x; xi[3] = b.y; }
        { const double2 a = __ldg(gi + 2), b = __ldg(gi + 3); yi[0] = a.x; yi[1] = a.y; yi[2] = b.x; yi[3] = b.y; }
        { const double2 a = __ldg(gi + 4), b = __ldg(gi + 5); zi[0] = a.x; zi[1] = a.y; zi[2] = b.x; zi[3] = b.y; }
        const uint32_t ig = i0 + 4u * tid;
        const uint32_t ig_warp = i0 + 4u * ((uint32_t)tid & ~31u);   // first i-particle of my warp
        const bool warp_idle = ig_warp >= (uint32_t)seg.ni;          // my warp holds padding only

        const bool masked = seg.same && (j0 < i0 + TI);
        const uint32_t n_stage = (j1 - j0 + kStageParticles - 1) / kStageParticles;
        const uint32_t s_begin = (masked && i0 > j0) ? (i0 - j0) / kStageParticles : 0;
        const double* jsrc = P.pk + ((size_t)seg.j_group + (j0 >> 2)) * kGroupFloats;
        const bool prune = (BOX == BOX_TRI) ? (range_ok && s_box->prune_ok != 0.0) : true;
        unsigned long long* const grow = P.out + (size_t)seg.hist * P.n_bins;     // MODE_GLOBAL: the result row itself
        OrthoRegs64 ob;
        if constexpr (BOX == BOX_ORTHO) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { ob.L[k] = s_box->L[k]; ob.invL[k] = s_box->invL[k]; }
        }

        if (tid == 0 && s_begin < n_stage) {
            const uint32_t b = stage_cnt & 1u;
            mbar_expect_tx(bar_addr + 8 * b, kStageBytes64);
            tma_load_1d(stage_addr + b * kStageBytes64, jsrc + (size_t)s_begin * kStageGroups * kGroupFloats, kStageBytes64, bar_addr + 8 * b);
        }
        for (uint32_t s = s_begin; s < n_stage; ++s) {
            const uint32_t b = stage_cnt & 1u;
            if (tid == 0 && s + 1 < n_stage) {
                const uint32_t nb = b ^ 1u;
                mbar_expect_tx(bar_addr + 8 * nb, kStageBytes64);
                tma_load_1d(stage_addr + nb * kStageBytes64, jsrc + (size_t)(s + 1) * kStageGroups * kGroupFloats, kStageBytes64, bar_addr + 8 * nb);
            }
            mbar_wait(bar_addr + 8 * b, (stage_cnt >> 1) & 1u);
            const double2* sj = reinterpret_cast<const double2*>(stage0 + b * (kStageBytes64 / 8));
            const uint32_t jbase = j0 + s * kStageParticles;
            const uint32_t n_grp = (SKIP && warp_idle) ? 0u : (min(j1 - jbase, (uint32_t)kStageParticles) + 3u) >> 2;
            const bool stage_masked = masked && (jbase < i0 + TI);
            // j-groups wholly below the diagonal for every lane of the warp are skipped, as is a padding-only warp
            auto body = [&](auto masked_c, const uint32_t g_begin) {
                constexpr bool MASKED = decltype(masked_c)::value;
#pragma unroll 1
                for (uint32_t g = g_begin; g < n_grp; ++g) {
                    const uint32_t jg = jbase + 4u * g;
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
                                if constexpr (PBOX) d2 = pair_d2_f64<BOX>(xi[r], yi[r], zi[r], xj[c], yj[c], zj[c], P.box0, ob, prune);
                                else d2 = pair_d2_f64<BOX>(xi[r], yi[r], zi[r], xj[c], yj[c], zj[c], *s_box, ob, prune);
                                bin_f64<MODE>(d2, P.rmax, P.scale, P.n_bins - 1u, hist_addr, cur_lo, cur_lim, trash_addr, keep, grow);
                            }
                    }
                }
            };
            if (stage_masked) body(std::true_type{}, (SKIP && ig_warp > jbase) ? min(n_grp, (ig_warp - jbase) >> 2) : 0u);
            else body(std::false_type{}, 0u);
            __syncthreads();
            ++stage_cnt;
        }
        __syncthreads();
    }
    flush();
}

}  // namespace cdh
