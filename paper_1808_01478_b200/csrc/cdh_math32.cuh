// cdh_math32.cuh -- the fp32 arithmetic policies of the tile kernel (cdh_sched.cuh): steps S2 distance, S3 minimum
// image, S4 bin and the S5 update of one j-group (4 j-particles x the thread's 4 i-particles = 16 pairs).
//
//   MathFast<BOX, TRI>    the production form: packed f32x2 arithmetic and the exact shortcuts of cdh_fast.cuh
//   MathSimple<BOX, VAR>  the pinned sequence spelled with the CUDA library's IEEE intrinsics (cross-validation,
//                         out-of-range fallback, and the aggregation variants behind flags)
// Both produce the same integers as the CPU oracle; they share no code with it.
#pragma once
#include "cdh_fast.cuh"

#ifndef CDH_TRI_RETEST
#define CDH_TRI_RETEST 1     // 1: the triclinic pruning margins are recomputed by the rare group that needs them instead of being kept in 16 registers (config 3: 753 -> 784 Gpairs/s)
#endif
#ifndef CDH_ONE_U
#define CDH_ONE_U 1     // 1: the second opaque 1.0f (TileParams::one_u) lives in a uniform register
#endif

namespace cdh {

struct ItemF32 {
    float xi[4], yi[4], zi[4];
};

__device__ __forceinline__ void load_i_group(const float* __restrict__ g, ItemF32& it) {
    const float4* gi = reinterpret_cast<const float4*>(g);
    const float4 XI = __ldg(gi), YI = __ldg(gi + 1), ZI = __ldg(gi + 2);
    it.xi[0] = XI.x; it.xi[1] = XI.y; it.xi[2] = XI.z; it.xi[3] = XI.w;
    it.yi[0] = YI.x; it.yi[1] = YI.y; it.yi[2] = YI.z; it.yi[3] = YI.w;
    it.zi[0] = ZI.x; it.zi[1] = ZI.y; it.zi[2] = ZI.z; it.zi[3] = ZI.w;
}

// TRI (BOX_TRI) additionally carries TRI_NOPRUNE: the definition (27 shifts) for every pair, in packed form -- the launch
// the host picks when r_max > h_min/2 or the box is too ill-conditioned for the pruning test (DESIGN.md "Triclinic
// pruning").  A kernel of its own so that the pruned kernel does not pay its registers (config 3: 76 bytes of spills).
constexpr int TRI_NOPRUNE = 8;

#ifndef CDH_TRI_FIXUP_WIDE
#define CDH_TRI_FIXUP_WIDE 0   // ... and not in the wide-range forms (config 3 shifted by up to 3 cells: 633 -> 621 Gpairs/s with it)
#endif
#ifndef CDH_TRI_FIXUP
#define CDH_TRI_FIXUP 4   // bit k: the narrow-range triclinic form k (TRI_GENERAL 0, TRI_UPPER 1, TRI_UPPER_B01 2) of the large-problem
                          // kernels bins first and moves the rare pair later.  Measured, 100,000 points: form 2 (config 3's) 821 -> 848
                          // Gpairs/s (ptxas parks the j-group in uniform registers across phase 2 and reads it from there in phase 1,
                          // and nothing of the rare path is merged back into the common one); form 0 656 -> 640, form 1 804 -> 774 and
                          // the SKIP kernels 508 -> 459 (they spill): left as they were
#endif

template <int BOX, int TRI>
struct MathFast {
    using Real = float;
    using Box = BoxConst;
    using Params = TileParams;
    static constexpr int kStageBytes = cdh::kStageBytes;
    static constexpr bool kPeriodic = BOX != BOX_NONE;
    static constexpr bool kHasClean = true;     // no box: coordinate extent; orthorhombic: full-range histogram; triclinic: d2 clamp
    static constexpr bool kCleanPadded = BOX == BOX_TRI;   // the clamp also drops NaN padding, the other two forms must not see any
    static constexpr int kUnroll = 1;
    static constexpr bool kNoPrune = BOX == BOX_TRI && (TRI & TRI_NOPRUNE) != 0;
    static constexpr int kTri = TRI & ~TRI_NOPRUNE;

    struct Launch {
        float prune_lim;        // triclinic: the zero-shift candidate decides while max_k |s_k - n_k| <= prune_lim
        bool clean;             // no box: every pinned d2 of the call is below the threshold and no coordinate is NaN
        Ones ones;
        f2 scale;
    };
    struct Item : ItemF32 {
        FastBox fb;
        uint32_t addr_c, sub_c;
        unsigned long long* grow;   // the result row, pinned in a register pair (MODE_GLOBAL / MODE_HYBRID): ptxas otherwise
                                    // rebuilds it from (out, row, n_bins) next to every reduction
    };

    __device__ __forceinline__ static bool launch_begin(const Params& P, Launch& L) {
        L.prune_lim = kPruneLimit;
        L.clean = false;
        if constexpr (BOX != BOX_NONE) {
            // The fast variants are exact only while the range of the fractional coordinates is small (fused rint and
            // exact B*n: n in {-1,0,1}; magic-number rint: |t| < 2^22).
            const float range = frac_range(P.range_keys);
            const bool mine = !(range <= P.range_lo) && (range <= P.range_hi || P.range_hi == __int_as_float(0x7f800000));
            if (!mine) return false;
            // TRI_WIDE: the error of s_k grows linearly with the range, and so must the margin (2x the 2^-17 of range 1.49)
            if constexpr (BOX == BOX_TRI && (TRI & TRI_WIDE) != 0) L.prune_lim = 0.5f - kPruneDelta * 2.0f * fmaxf(1.0f, range * (1.0f / 1.49f));
            // orthorhombic, fractional range <= 1.49: every wrapped component is within L/2 (1 + 2^-18), so the host could size
            // the private histogram for every reachable distance (keep_bins != 0); no NaN coordinate in the call
            if constexpr (BOX == BOX_ORTHO) L.clean = P.keep_bins != 0u && __ldg(P.range_keys + 6) == 0u;
            // triclinic: the host found that the slot of bin(thr2) is not a flushed one: dropped pairs are clamped into it
            if constexpr (BOX == BOX_TRI) L.clean = P.keep_bins != 0u;
        } else {
            L.clean = __float_as_uint(coord_extent2_ru(P.range_keys)) < P.thr2_bits;
        }
        L.ones.r = dup2(P.one); L.ones.u = CDH_ONE_U ? dup2(P.one_u) : L.ones.r;
        L.scale = dup2(P.scale);
        return true;
    }

    template <int MODE>
    __device__ __forceinline__ static void key_begin(const Params& P, const Launch&, const Seg& seg, HistView& hv) {
        if constexpr (MODE == MODE_HYBRID) {
            hv.lo = min(__ldg(P.win_lo + seg.hist), P.n_bins - min(P.n_bins, P.smem_bins));
            hv.lim = min(P.smem_bins, P.n_bins - hv.lo);
        } else {
            hv.lo = seg.bin_lo; hv.lim = seg.bin_cnt + seg.last_sweep;
            if constexpr (BOX != BOX_NONE && MODE == MODE_SHARED) if (P.keep_bins != 0u) hv.lim = P.keep_bins;   // slots beyond: dropped pairs
        }
    }

    __device__ __forceinline__ static void item_begin(const Params&, const Launch&, const float* __restrict__ gi,
                                                      const Box* s_box, const HistView& hv, Item& it) {
        load_i_group(gi, it);
        if constexpr (BOX == BOX_ORTHO) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { it.fb.L[k] = s_box->L[k]; it.fb.invL[k] = (TRI == ORTHO_FUSED) ? s_box->invLf[k] : s_box->invL[k]; }
        }
        if constexpr (BOX == BOX_TRI) {
#pragma unroll
            for (int k = 0; k < 9; ++k) { it.fb.B[k] = s_box->B[k]; it.fb.Binv[k] = s_box->Binv[k]; }
        }
        // pinned in a register each (as grow): where registers are short ptxas otherwise rebuilds the address constant from
        // the stage count and the CTA's shared window in every group (8 instructions per 16 pairs in the triclinic kernels)
        asm volatile("mov.b32 %0, %1;" : "=r"(it.addr_c) : "r"(hv.hist_addr - 4u * (kFloorMagicBits + hv.lo)));
        it.sub_c = kFloorMagicBits + hv.lo;
        asm volatile("mov.b64 %0, %1;" : "=l"(it.grow) : "l"(hv.grow));
    }

    template <int MODE, int KIND, bool SKIPV = false>
    __device__ __forceinline__ static void group(const Params& P, const Launch& L, const Item& it, const unsigned char* stage,
                                                 uint32_t g, uint32_t jg, uint32_t ig, const HistView& hv, const Box* s_box) {
        constexpr bool MASKED = KIND == KIND_MASKED;
        constexpr bool CLEAN = KIND == KIND_CLEAN && (MODE == MODE_SHARED || MODE == MODE_HYBRID || MODE == MODE_GLOBAL);
        constexpr bool FIXUP = BOX == BOX_TRI && MODE == MODE_SHARED && !SKIPV && (CDH_TRI_FIXUP_WIDE || (kTri & TRI_WIDE) == 0) && (CDH_TRI_FIXUP & (1 << (kTri & 3))) != 0;
        const float4* sj = reinterpret_cast<const float4*>(stage);
        const float4 XJ = sj[3 * g], YJ = sj[3 * g + 1], ZJ = sj[3 * g + 2];
        const f2 XA = pk2(XJ.x, XJ.y), XB = pk2(XJ.z, XJ.w), YA = pk2(YJ.x, YJ.y), YB = pk2(YJ.z, YJ.w),
                 ZA = pk2(ZJ.x, ZJ.y), ZB = pk2(ZJ.z, ZJ.w);
        // phase 1: the 16 squared distances of this j-group, branch free
        f2 D2[kR][2];
        if constexpr (kNoPrune) {
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                D2[r][0] = pair_d2_full_packed<kTri>(XA, YA, ZA, it.xi[r], it.yi[r], it.zi[r], it.fb, s_box, L.ones);
                D2[r][1] = pair_d2_full_packed<kTri>(XB, YB, ZB, it.xi[r], it.yi[r], it.zi[r], it.fb, s_box, L.ones);
            }
        } else {
#if CDH_TRI_RETEST
            // the per-element pruning margins are NOT kept: only their maximum over the group; the rare group that needs the
            // search recomputes them (16 floats fewer live across phase 1)
            [[maybe_unused]] float fm_all = 0.0f;
#pragma unroll
            for (int r = 0; r < kR; ++r) {
#pragma unroll
                for (int hlf = 0; hlf < 2; ++hlf) {
                    float f0, f1;
                    D2[r][hlf] = pair_d2_fast<BOX, kTri>(hlf ? XB : XA, hlf ? YB : YA, hlf ? ZB : ZA, it.xi[r], it.yi[r], it.zi[r],
                                                         it.fb, L.ones, f0, f1);
                    if constexpr (BOX == BOX_TRI) fm_all = fmaxf(fmaxf(fm_all, f0), f1);
                }
            }
            if constexpr (FIXUP) {
                // Shared-memory histogram: bin the whole group first, with the d2 of the first-guess image, and MOVE the rare
                // pair the neighbour search corrects afterwards (-1 on the slot it went to, +1 on the right one).  The common
                // path then carries nothing of the rare one: corrected values merged back into D2 cost it 12 MOV per group.
                constexpr bool CLEANF = CLEAN;
#pragma unroll
                for (int r = 0; r < kR; ++r) {
#pragma unroll
                    for (int hlf = 0; hlf < 2; ++hlf) {
                        bool k0 = true, k1 = true;
                        if constexpr (MASKED) { k0 = jg + 2 * hlf > ig + r; k1 = jg + 2 * hlf + 1 > ig + r; }
                        bin_fast2<MODE, CLEANF, true>(D2[r][hlf], k0, k1, L.scale, L.ones.r, P.thr2_bits, it.addr_c, it.sub_c, hv, it.grow);
                    }
                }
                if (fm_all > L.prune_lim) {
                    const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
                    for (int r = 0; r < kR; ++r) {
#pragma unroll
                        for (int hlf = 0; hlf < 2; ++hlf) {
                            float xr = it.xi[r], f0, f1;
                            asm volatile("" : "+f"(xr));                 // opaque: recomputed here, nothing of phase 1 is kept alive
                            const f2 d2f = pair_d2_fast<BOX, kTri>(hlf ? XB : XA, hlf ? YB : YA, hlf ? ZB : ZA, xr, it.yi[r], it.zi[r], it.fb, L.ones, f0, f1);
                            float pf, qf; upk2(d2f, pf, qf);
                            bool k0 = true, k1 = true;
                            if constexpr (MASKED) { k0 = jg + 2 * hlf > ig + r; k1 = jg + 2 * hlf + 1 > ig + r; }
                            if (f0 > L.prune_lim && k0) {
                                const float pe = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf], yj[2 * hlf], zj[2 * hlf], s_box);
                                const uint32_t a_old = bin_addr_shared<CLEANF, true>(pf, k0, L.scale, L.ones.r, P.thr2_bits, it.addr_c, hv);
                                const uint32_t a_new = bin_addr_shared<CLEANF, true>(pe, k0, L.scale, L.ones.r, P.thr2_bits, it.addr_c, hv);
                                if (a_old != a_new) { hist_add(a_old, 0xFFFFFFFFu); hist_inc(a_new); }
                            }
                            if (f1 > L.prune_lim && k1) {
                                const float qe = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf + 1], yj[2 * hlf + 1], zj[2 * hlf + 1], s_box);
                                const uint32_t a_old = bin_addr_shared<CLEANF, true>(qf, k1, L.scale, L.ones.r, P.thr2_bits, it.addr_c, hv);
                                const uint32_t a_new = bin_addr_shared<CLEANF, true>(qe, k1, L.scale, L.ones.r, P.thr2_bits, it.addr_c, hv);
                                if (a_old != a_new) { hist_add(a_old, 0xFFFFFFFFu); hist_inc(a_new); }
                            }
                        }
                    }
                }
                return;
            } else if constexpr (BOX == BOX_TRI) {
                if (fm_all > L.prune_lim) {
                    const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
                    for (int r = 0; r < kR; ++r) {
#pragma unroll
                        for (int hlf = 0; hlf < 2; ++hlf) {
                            float xr = it.xi[r], f0, f1;
                            asm volatile("" : "+f"(xr));                 // opaque: the margins are recomputed, not kept alive
                            (void)pair_d2_fast<BOX, kTri>(hlf ? XB : XA, hlf ? YB : YA, hlf ? ZB : ZA, xr, it.yi[r], it.zi[r], it.fb, L.ones, f0, f1);
                            float p, q; upk2(D2[r][hlf], p, q);
                            bool n0 = f0 > L.prune_lim, n1 = f1 > L.prune_lim;
                            if constexpr (MASKED) { n0 = n0 && (jg + 2 * hlf > ig + r); n1 = n1 && (jg + 2 * hlf + 1 > ig + r); }
                            if (n0) p = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf], yj[2 * hlf], zj[2 * hlf], s_box);
                            if (n1) q = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf + 1], yj[2 * hlf + 1], zj[2 * hlf + 1], s_box);
                            D2[r][hlf] = pk2(p, q);
                        }
                    }
                }
            }
#else
            float fm[kR][2][2];
            [[maybe_unused]] float fm_all = 0.0f;
#pragma unroll
            for (int r = 0; r < kR; ++r) {
#pragma unroll
                for (int hlf = 0; hlf < 2; ++hlf) {
                    D2[r][hlf] = pair_d2_fast<BOX, kTri>(hlf ? XB : XA, hlf ? YB : YA, hlf ? ZB : ZA, it.xi[r], it.yi[r], it.zi[r],
                                                         it.fb, L.ones, fm[r][hlf][0], fm[r][hlf][1]);
                    if constexpr (BOX == BOX_TRI) fm_all = fmaxf(fmaxf(fm_all, fm[r][hlf][0]), fm[r][hlf][1]);
                }
            }
            if constexpr (BOX == BOX_TRI) {
                if (fm_all > L.prune_lim) {
                    // rare: some element of the group has a fractional coordinate within kPruneDelta of +-1/2: run the
                    // definition for those elements, out of line
                    const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
                    for (int r = 0; r < kR; ++r) {
#pragma unroll
                        for (int hlf = 0; hlf < 2; ++hlf) {
                            float p, q; upk2(D2[r][hlf], p, q);
                            bool n0 = fm[r][hlf][0] > L.prune_lim, n1 = fm[r][hlf][1] > L.prune_lim;
                            if constexpr (MASKED) { n0 = n0 && (jg + 2 * hlf > ig + r); n1 = n1 && (jg + 2 * hlf + 1 > ig + r); }
                            if (n0) p = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf], yj[2 * hlf], zj[2 * hlf], s_box);
                            if (n1) q = tri_full_d2(it.xi[r], it.yi[r], it.zi[r], xj[2 * hlf + 1], yj[2 * hlf + 1], zj[2 * hlf + 1], s_box);
                            D2[r][hlf] = pk2(p, q);
                        }
                    }
                }
            }
#endif
        }
        // phase 2: bin and update
#pragma unroll
        for (int r = 0; r < kR; ++r) {
#pragma unroll
            for (int hlf = 0; hlf < 2; ++hlf) {
                bool k0 = true, k1 = true;
                if constexpr (MASKED) { k0 = jg + 2 * hlf > ig + r; k1 = jg + 2 * hlf + 1 > ig + r; }
                bin_fast2<MODE, CLEAN && (BOX != BOX_TRI || MODE == MODE_SHARED), BOX == BOX_TRI>(D2[r][hlf], k0, k1, L.scale, L.ones.r, P.thr2_bits, it.addr_c, it.sub_c, hv, it.grow);
            }
        }
    }
};

template <int BOX, int VAR>
struct MathSimple {
    using Real = float;
    using Box = BoxConst;
    using Params = TileParams;
    static constexpr int kStageBytes = cdh::kStageBytes;
    static constexpr bool kPeriodic = BOX != BOX_NONE;
    static constexpr bool kHasClean = false;
    static constexpr bool kCleanPadded = false;
    static constexpr int kUnroll = 1;
    struct Launch { bool clean; };
    using Item = ItemF32;

    __device__ __forceinline__ static bool launch_begin(const Params& P, Launch& L) {
        L.clean = false;
        if constexpr (BOX != BOX_NONE) {
            const float range = frac_range(P.range_keys);
            return !(range <= P.range_lo) && (range <= P.range_hi || P.range_hi == __int_as_float(0x7f800000));
        }
        return true;
    }
    template <int MODE>
    __device__ __forceinline__ static void key_begin(const Params&, const Launch&, const Seg& seg, HistView& hv) {
        hv.lo = seg.bin_lo; hv.lim = seg.bin_cnt + seg.last_sweep;
    }
    __device__ __forceinline__ static void item_begin(const Params&, const Launch&, const float* __restrict__ gi, const Box*,
                                                      const HistView&, Item& it) {
        load_i_group(gi, it);
    }
    template <int MODE, int KIND, bool SKIPV = false>
    __device__ __forceinline__ static void group(const Params& P, const Launch&, const Item& it, const unsigned char* stage,
                                                 uint32_t g, uint32_t jg, uint32_t ig, const HistView& hv, const Box* s_box) {
        constexpr bool MASKED = KIND == KIND_MASKED;
        const float4* sj = reinterpret_cast<const float4*>(stage);
        const float4 XJ = sj[3 * g], YJ = sj[3 * g + 1], ZJ = sj[3 * g + 2];
        const float xj[4] = {XJ.x, XJ.y, XJ.z, XJ.w}, yj[4] = {YJ.x, YJ.y, YJ.z, YJ.w}, zj[4] = {ZJ.x, ZJ.y, ZJ.z, ZJ.w};
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int r = 0; r < kR; ++r) {
                const bool keep = !MASKED || (jg + c > ig + r);
                const float d2 = pair_d2_simple<BOX>(it.xi[r], it.yi[r], it.zi[r], xj[c], yj[c], zj[c], s_box);
                bin_simple<VAR, MODE>(d2, keep, P.rmax, P.scale, P.n_bins, hv.hist_addr, hv.lo, hv.lim, hv.grow);
            }
    }
};

}  // namespace cdh
