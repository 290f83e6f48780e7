// cdh_tile.cuh -- K1: the persistent tile kernel (steps S1-S7 of SURVEY.md 8a).
//
// One CTA owns one private uint32 histogram in shared memory (histogram strategy 3, PAPER.md:117-123,
// and the paper's shared-memory kernel) and pulls work items (i-tile, j-chunk) from a
// global counter.  Items are ordered by (histogram row, bin sweep), so a CTA flushes into the uint64
// result only when that key changes, when its increment budget nears 2^32 and at exit.
// Each thread keeps R = 4 i-particles in registers; the j-chunk streams through two 3 KB shared-memory
// stages filled by 1-D TMA bulk copies (cp.async.bulk + mbarrier); all lanes read the same j-group
// (LDS.128 broadcast).  Intra-species segments only schedule j-chunks that reach above the diagonal
// (triangular schedule, Fig. 1, 223-225); tiles on the diagonal take the masked path.
#pragma once
#include <type_traits>
#include "cdh_fast.cuh"

#ifndef CDH_GUNROLL
#define CDH_GUNROLL 1      // j-groups unrolled in the inner loop (2 was measured: cfg2 -0.4 %, cfg5 -1.6 %, cfg3 +1.4 %)
#endif


namespace cdh {

constexpr int kGUnroll = CDH_GUNROLL;
constexpr int kR = 4;                       // i-particles per thread (one group)
constexpr int kSmemHeader = 128;            // mbarriers + scheduler slot
constexpr uint64_t kMaxIncrements = 0xFFFFFFFFull;

__host__ __device__ constexpr int tile_smem_bytes(int smem_bins) {
    return kSmemHeader + 2 * kStageBytes + sizeof(BoxConst) + 16 + 4 * (smem_bins + 2);   // + Q3 slot + trash slot
}

// SKIP: a warp skips the j-groups that lie below the diagonal for all of its lanes, and every group if it holds only
// padding i-particles (ragged last i-tile).  For frames of small species (a few i-tiles each) this is up to 44 % of a
// diagonal block and half of a ragged tile; the host takes these variants only then (cdh_api.cu), because the warp-dependent
// trip count costs the large-problem kernels 2-5 % (measured: config 2 1258 -> 1221, config 5 1914 -> 1816 Gpairs/s).
template <int BOX, int TRI, int T, int VAR, int MODE, int MINB, bool SKIP = false>
__global__ void __launch_bounds__(T, MINB) tile_kernel(const TileParams P) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int TI = T * kR;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    volatile uint32_t* s_item = reinterpret_cast<volatile uint32_t*>(smem + 16);
    float* stage0 = reinterpret_cast<float*>(smem + kSmemHeader);
    BoxConst* s_box = reinterpret_cast<BoxConst*>(smem + kSmemHeader + 2 * kStageBytes);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + kSmemHeader + 2 * kStageBytes + sizeof(BoxConst) + 16);
    const uint32_t hist_addr = smem_u32(s_hist);
    const uint32_t bar_addr = smem_u32(bars);
    const uint32_t stage_addr = smem_u32(stage0);
    const int tid = threadIdx.x;

    // The fast variants are exact only while the range of the fractional coordinates is small (fused rint and
    // exact B*n: n in {-1,0,1}; magic-number rint: |t| < 2^22).  Every launch of the call reads the range the
    // repack kernel measured and exactly one of them does the work (no host synchronisation).  Uniform over the grid.
    float prune_lim = kPruneLimit;          // triclinic: the zero-shift candidate decides while max_k |s_k - n_k| <= prune_lim
    if constexpr (BOX != BOX_NONE) {
        const float range = frac_range(P.range_keys);
        const bool mine = !(range <= P.range_lo) && (range <= P.range_hi || P.range_hi == __int_as_float(0x7f800000));
        if (!mine) return;
        // TRI_WIDE: the error of s_k grows linearly with the range, and so must the margin (2x the 2^-17 of range 1.49)
        if constexpr (BOX == BOX_TRI && (TRI & TRI_WIDE) != 0) prune_lim = 0.5f - kPruneDelta * 2.0f * fmaxf(1.0f, range * (1.0f / 1.49f));
    }

    if (tid == 0) { mbar_init(bar_addr, 1); mbar_init(bar_addr + 8, 1); fence_mbar_init(); }
    for (uint32_t b = tid; b <= P.smem_bins + 1; b += T) s_hist[b] = 0;
    const uint32_t trash_addr = hist_addr + 4u * (P.smem_bins + 1u);   // never flushed
    __syncthreads();

    uint32_t stage_cnt = 0;                 // stages consumed so far: buffer = cnt & 1, parity = (cnt >> 1) & 1
    uint32_t cur_key = 0xFFFFFFFFu, cur_hist = 0, cur_lo = 0, cur_lim = 0, cur_box = 0xFFFFFFFFu;
    uint64_t increments = 0;                // upper bound of increments since the last flush
    const f2 ONE = dup2(P.one);
    const f2 SCALE = dup2(P.scale);

    auto flush = [&]() {
        __syncthreads();
        if (MODE != MODE_GLOBAL && cur_key != 0xFFFFFFFFu) {
            unsigned long long* o = P.out + (size_t)cur_hist * P.n_bins;
            for (uint32_t b = tid; b < cur_lim; b += T) {
                const uint32_t v = s_hist[b];
                if (v) {
                    s_hist[b] = 0;
                    atomicAdd(o + min(cur_lo + b, P.n_bins - 1u), (unsigned long long)v);   // Q3 slot -> last bin
                }
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

        // row of the item: largest r with rows[r].item_prefix <= item
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
            const float* src = reinterpret_cast<const float*>(P.boxes + seg.box);
            for (int k = tid; k < (int)(sizeof(BoxConst) / 4); k += T) reinterpret_cast<float*>(s_box)[k] = __ldg(src + k);
            cur_box = seg.box;
            __syncthreads();
        }

        // my R = 4 i-particles: one group
        const float4* gi = reinterpret_cast<const float4*>(P.pk + ((size_t)seg.i_group + (i0 >> 2) + tid) * kGroupFloats);
        const float4 XI = __ldg(gi), YI = __ldg(gi + 1), ZI = __ldg(gi + 2);
        const float xi[4] = {XI.x, XI.y, XI.z, XI.w}, yi[4] = {YI.x, YI.y, YI.z, YI.w}, zi[4] = {ZI.x, ZI.y, ZI.z, ZI.w};
        const uint32_t ig = i0 + 4u * tid;          // index of my first i-particle inside the species
        const uint32_t ig_warp = i0 + 4u * ((uint32_t)tid & ~31u);   // first i-particle of my warp (128 consecutive ones)
        const bool warp_idle = ig_warp >= (uint32_t)seg.ni;          // ragged last i-tile: my warp holds padding only

        const bool masked = seg.same && (j0 < i0 + TI);       // some j <= some i: test j > i per pair
        const uint32_t n_stage = (j1 - j0 + kStageParticles - 1) / kStageParticles;
        const uint32_t s_begin = (masked && i0 > j0) ? (i0 - j0) / kStageParticles : 0;   // stages wholly below the diagonal
        const float* jsrc = P.pk + ((size_t)seg.j_group + (j0 >> 2)) * kGroupFloats;

        FastBox fb;
        if constexpr (VAR == VAR_FAST && BOX == BOX_ORTHO) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { fb.L[k] = s_box->L[k]; fb.invL[k] = (TRI == ORTHO_FUSED) ? s_box->invLf[k] : s_box->invL[k]; }
        }
        if constexpr (VAR == VAR_FAST && BOX == BOX_TRI) {
#pragma unroll
            for (int k = 0; k < 9; ++k) { fb.B[k] = s_box->B[k]; fb.Binv[k] = s_box->Binv[k]; }
        }
        const bool prune = (BOX == BOX_TRI) ? (s_box->prune_ok != 0.0f) : true;
        const uint32_t addr_c = hist_addr - 4u * (kFloorMagicBits + cur_lo);
        const uint32_t sub_c = kFloorMagicBits + cur_lo;
        unsigned long long* const grow = P.out + (size_t)seg.hist * P.n_bins;     // MODE_GLOBAL: the result row itself

        if (tid == 0 && s_begin < n_stage) {
            const uint32_t b = stage_cnt & 1u;
            mbar_expect_tx(bar_addr + 8 * b, kStageBytes);
            tma_load_1d(stage_addr + b * kStageBytes, jsrc + (size_t)s_begin * kStageGroups * kGroupFloats, kStageBytes, bar_addr + 8 * b);
        }
        for (uint32_t s = s_begin; s < n_stage; ++s) {
            const uint32_t b = stage_cnt & 1u;
            if (tid == 0 && s + 1 < n_stage) {
                const uint32_t nb = b ^ 1u;
                mbar_expect_tx(bar_addr + 8 * nb, kStageBytes);
                tma_load_1d(stage_addr + nb * kStageBytes, jsrc + (size_t)(s + 1) * kStageGroups * kGroupFloats, kStageBytes, bar_addr + 8 * nb);
            }
            mbar_wait(bar_addr + 8 * b, (stage_cnt >> 1) & 1u);
            const float4* sj = reinterpret_cast<const float4*>(stage0 + b * (kStageBytes / 4));
            const uint32_t jbase = j0 + s * kStageParticles;                   // species index of the stage's first j
            const uint32_t n_grp = (SKIP && warp_idle) ? 0u : (min(j1 - jbase, (uint32_t)kStageParticles) + 3u) >> 2;

            // only stages that touch the diagonal band need the mask
            const bool stage_masked = masked && (jbase < i0 + TI);
            auto body = [&](auto masked_c, const uint32_t g_begin) {
                constexpr bool MASKED = decltype(masked_c)::value;
#pragma unroll kGUnroll
                for (uint32_t g = g_begin; g < n_grp; ++g) {
                    const float4 XJ = sj[3 * g], YJ = sj[3 * g + 1], ZJ = sj[3 * g + 2];
                    const uint32_t jg = jbase + 4u * g;
                    if constexpr (VAR != VAR_FAST) {
                        const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
                        for (int c = 0; c < 4; ++c)
#pragma unroll
                            for (int r = 0; r < kR; ++r) {
                                const bool keep = !MASKED || (jg + c > ig + r);
                                const float d2 = pair_d2_simple<BOX>(xi[r], yi[r], zi[r], xj[c], yj[c], zj[c], s_box);
                                bin_simple<VAR, MODE>(d2, keep, P.rmax, P.scale, P.n_bins, hist_addr, cur_lo, cur_lim, grow);
                            }
                    } else {
                        const f2 XA = pk2(XJ.x, XJ.y), XB = pk2(XJ.z, XJ.w), YA = pk2(YJ.x, YJ.y), YB = pk2(YJ.z, YJ.w),
                                 ZA = pk2(ZJ.x, ZJ.y), ZB = pk2(ZJ.z, ZJ.w);
                        // phase 1: the 16 squared distances of this j-group, branch free
                        f2 D2[kR][2];
                        float fm[kR][2][2];
                        [[maybe_unused]] float fm_all = 0.0f;
#pragma unroll
                        for (int r = 0; r < kR; ++r) {
#pragma unroll
                            for (int hlf = 0; hlf < 2; ++hlf) {
                                D2[r][hlf] = pair_d2_fast<BOX, TRI>(hlf ? XB : XA, hlf ? YB : YA, hlf ? ZB : ZA, xi[r], yi[r], zi[r],
                                                                    fb, ONE, fm[r][hlf][0], fm[r][hlf][1]);
                                if constexpr (BOX == BOX_TRI) fm_all = fmaxf(fmaxf(fm_all, fm[r][hlf][0]), fm[r][hlf][1]);
                            }
                        }
                        if constexpr (BOX == BOX_TRI) {
                            if (!prune) {
                                // pruning is off for this box / r_max: the definition for every pair, packed
#pragma unroll
                                for (int r = 0; r < kR; ++r) {
                                    D2[r][0] = pair_d2_full_packed<TRI>(XA, YA, ZA, xi[r], yi[r], zi[r], fb, s_box, ONE);
                                    D2[r][1] = pair_d2_full_packed<TRI>(XB, YB, ZB, xi[r], yi[r], zi[r], fb, s_box, ONE);
                                }
                            } else if (fm_all > prune_lim) {
                                // rare: some element of the group has a fractional coordinate within kPruneDelta of
                                // +-1/2: run the definition for those elements, out of line
                                const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
                                for (int r = 0; r < kR; ++r) {
#pragma unroll
                                    for (int hlf = 0; hlf < 2; ++hlf) {
                                        float p, q; upk2(D2[r][hlf], p, q);
                                        bool n0 = fm[r][hlf][0] > prune_lim, n1 = fm[r][hlf][1] > prune_lim;
                                        if constexpr (MASKED) { n0 = n0 && (jg + 2 * hlf > ig + r); n1 = n1 && (jg + 2 * hlf + 1 > ig + r); }
                                        if (n0) p = tri_full_d2(xi[r], yi[r], zi[r], xj[2 * hlf], yj[2 * hlf], zj[2 * hlf], s_box);
                                        if (n1) q = tri_full_d2(xi[r], yi[r], zi[r], xj[2 * hlf + 1], yj[2 * hlf + 1], zj[2 * hlf + 1], s_box);
                                        D2[r][hlf] = pk2(p, q);
                                    }
                                }
                            }
                        }
                        // phase 2: bin and update
#pragma unroll
                        for (int r = 0; r < kR; ++r) {
#pragma unroll
                            for (int hlf = 0; hlf < 2; ++hlf) {
                                bool k0 = true, k1 = true;
                                if constexpr (MASKED) { k0 = jg + 2 * hlf > ig + r; k1 = jg + 2 * hlf + 1 > ig + r; }
                                bin_fast2<MODE>(D2[r][hlf], k0, k1, SCALE, ONE, P.thr2_bits, addr_c, hist_addr, sub_c, cur_lim, trash_addr, grow, P.n_bins - 1u);
                            }
                        }
                    }
                }
            };
            if (stage_masked) body(std::true_type{}, (SKIP && ig_warp > jbase) ? min(n_grp, (ig_warp - jbase) >> 2) : 0u);
            else body(std::false_type{}, 0u);

            __syncthreads();          // everyone is done with buffer b before it is refilled
            ++stage_cnt;
        }
        __syncthreads();              // s_item is rewritten at the top of the loop
    }
    flush();
}

}  // namespace cdh
