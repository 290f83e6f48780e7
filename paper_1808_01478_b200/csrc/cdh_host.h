// cdh_host.h -- host-side logic of libcdh: argument validation, fp32 constants derived in double,
// the exact d2 threshold, the bin-sweep plan and the work tables (segments and rows).  Plain C++,
// no CUDA calls.  Must be compiled without FP contraction (-ffp-contract=off): the constants are part
// of the pinned sequence.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include "cdh_device.cuh"
#include "cdh_f64.cuh"
#include "../../include/cdh.h"

namespace cdh {

inline uint32_t f32_bits(float x) { uint32_t u; std::memcpy(&u, &x, 4); return u; }
inline float bits_f32(uint32_t u) { float x; std::memcpy(&x, &u, 4); return x; }

// Smallest fp32 x >= 0 whose correctly rounded square root is >= rmax (sqrtf is correctly rounded and
// monotone): "d < rmax" <=> "bits(d2) < bits(x)" for d2 >= +0.
inline uint32_t d2_threshold_bits(float rmax) {
    float x = (float)((double)rmax * (double)rmax);
    if (!(x <= 3.0e38f)) return 0x7f800000u;                 // r_max^2 overflows: only inf / NaN are dropped
    while (x > 0.0f && sqrtf(std::nextafterf(x, 0.0f)) >= rmax) x = std::nextafterf(x, 0.0f);
    while (sqrtf(x) < rmax) x = std::nextafterf(x, INFINITY);
    return f32_bits(x);
}

// b (columns = box vectors) and b^-1 = adj(b)/det(b) in double with a fixed parenthesisation; API rows
// are the box vectors (Eq. 5; reading Q6).  Returns false if singular / non-finite.
inline bool box_matrices(const double* box9, double B[9], double Bi[9], double* h_min) {
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) B[3 * r + c] = box9[3 * c + r];
    const double b00 = B[0], b01 = B[1], b02 = B[2], b10 = B[3], b11 = B[4], b12 = B[5], b20 = B[6], b21 = B[7], b22 = B[8];
    const double det = b00 * (b11 * b22 - b12 * b21) - b01 * (b10 * b22 - b12 * b20) + b02 * (b10 * b21 - b11 * b20);
    if (!std::isfinite(det) || det == 0.0) return false;
    Bi[0] = (b11 * b22 - b12 * b21) / det;  Bi[1] = -(b01 * b22 - b02 * b21) / det;  Bi[2] = (b01 * b12 - b02 * b11) / det;
    Bi[3] = -(b10 * b22 - b12 * b20) / det; Bi[4] = (b00 * b22 - b02 * b20) / det;   Bi[5] = -(b00 * b12 - b02 * b10) / det;
    Bi[6] = (b10 * b21 - b11 * b20) / det;  Bi[7] = -(b00 * b21 - b01 * b20) / det;  Bi[8] = (b00 * b11 - b01 * b10) / det;
    double hm = INFINITY;
    for (int k = 0; k < 3; ++k) {                             // height k = 1 / |row k of b^-1|
        const double n = std::sqrt(Bi[3 * k] * Bi[3 * k] + Bi[3 * k + 1] * Bi[3 * k + 1] + Bi[3 * k + 2] * Bi[3 * k + 2]);
        if (!std::isfinite(n) || n == 0.0) return false;
        hm = std::fmin(hm, 1.0 / n);
    }
    for (int k = 0; k < 9; ++k) if (!std::isfinite(Bi[k])) return false;
    *h_min = hm;
    return true;
}

// Fused rint: the pinned form n = rint(fl(d * invL)) switches from n = 0 to n = 1 at the
// float c_half = max{c : fl(c * invL) <= 1/2}; the fused form rint(d * invLf) (exact product, one rounding at integer
// granularity, ties to even) switches at max{c : c * invLf <= 1/2}.  Search the neighbours of invL for an invLf whose
// switch point is the same float; then both forms agree for every |d| below the 3/2 switch (the kernel's range
// limit 1.49 keeps |d * invL| well below it).  Products of two floats are exact in double.
inline bool fused_rint_constant(float invL, float* invLf) {
    if (!(invL > 0.0f) || !std::isfinite(invL)) return false;
    auto pinned_zero = [&](float c) { return (float)((double)c * (double)invL) <= 0.5f; };
    float c = (float)(0.5 / (double)invL);
    if (!std::isfinite(c) || !(c > 0.0f)) return false;
    for (int it = 0; it < 64 && !pinned_zero(c); ++it) c = std::nextafterf(c, 0.0f);
    for (int it = 0; it < 64 && pinned_zero(std::nextafterf(c, INFINITY)); ++it) c = std::nextafterf(c, INFINITY);
    if (!pinned_zero(c) || pinned_zero(std::nextafterf(c, INFINITY))) return false;
    const float c_next = std::nextafterf(c, INFINITY);
    for (int d = 0; d <= 8; ++d)
        for (int sgn = 1; sgn >= -1; sgn -= 2) {
            const float cand = bits_f32(f32_bits(invL) + (uint32_t)(sgn * d));
            if (!(cand > 0.0f) || !std::isfinite(cand)) continue;
            if ((double)c * (double)cand <= 0.5 && !((double)c_next * (double)cand <= 0.5)) { *invLf = cand; return true; }
        }
    return false;
}

// Fills one BoxConst.  Returns false on an invalid box.
inline bool make_box_const(int box_type, const double* box9, double r_max, BoxConst* bc) {
    std::memset(bc, 0, sizeof *bc);
    if (box_type == CDH_BOX_ORTHO) {
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) {
                const double v = box9[3 * r + c];
                if (!std::isfinite(v)) return false;
                if (r != c && v != 0.0) return false;
                if (r == c && v == 0.0) return false;
            }
        for (int c = 0; c < 3; ++c) {
            bc->L[c] = (float)box9[4 * c];
            bc->invL[c] = (float)(1.0 / box9[4 * c]);
            if (!std::isfinite(bc->invL[c]) || bc->L[c] == 0.0f) return false;
        }
        // prune_ok doubles as "fused rint available" for ORTHO (negative box lengths take the plain form)
        bc->prune_ok = 1.0f;
        for (int c = 0; c < 3; ++c)
            if (!fused_rint_constant(bc->invL[c], &bc->invLf[c])) { bc->invLf[c] = bc->invL[c]; bc->prune_ok = 0.0f; }
    } else if (box_type == CDH_BOX_TRICLINIC) {
        for (int k = 0; k < 9; ++k) if (!std::isfinite(box9[k])) return false;
        double B[9], Bi[9], h_min;
        if (!box_matrices(box9, B, Bi, &h_min)) return false;
        for (int k = 0; k < 9; ++k) { bc->B[k] = (float)B[k]; bc->Binv[k] = (float)Bi[k]; }
        int m = 0;
        for (int i = -1; i <= 1; ++i)
            for (int j = -1; j <= 1; ++j)
                for (int k = -1; k <= 1; ++k, ++m)
                    for (int r = 0; r < 3; ++r)
                        bc->S[m][r] = ((float)i * bc->B[3 * r] + (float)j * bc->B[3 * r + 1]) + (float)k * bc->B[3 * r + 2];
        // The zero-shift candidate alone decides when r_max <= h_min/2 and the kernel's
        // fractional-coordinate test (|s_k - n_k| <= 1/2 - 2^-17) is trustworthy, i.e. the fp32 error of s_k stays
        // below 2^-18 for |fractional differences| <= 1.5 (the range limit of the fast path is 1.49): that error is
        // bounded by 15 * 2^-24 * kappa, kappa = max_k sum_c sum_m |Binv[k][c]| |B[c][m]|.
        double kappa = 0.0;
        for (int k = 0; k < 3; ++k) {
            double row = 0.0;
            for (int c = 0; c < 3; ++c)
                for (int m = 0; m < 3; ++m) row += std::fabs(Bi[3 * k + c]) * std::fabs(B[3 * c + m]);
            kappa = std::fmax(kappa, row);
        }
        const bool margin_ok = 15.0 * kappa * std::ldexp(1.0, -24) <= std::ldexp(1.0, -18);
        bc->prune_ok = (r_max <= 0.5 * h_min * (1.0 + 1e-9) && margin_ok) ? 1.0f : 0.0f;
    }
    return true;
}

// The same constants for the double-precision path (T = double: no rounding after the double derivation).
inline bool make_box_const64(int box_type, const double* box9, double r_max, BoxConst64* bc) {
    std::memset(bc, 0, sizeof *bc);
    if (box_type == CDH_BOX_ORTHO) {
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) {
                const double v = box9[3 * r + c];
                if (!std::isfinite(v)) return false;
                if (r != c && v != 0.0) return false;
                if (r == c && v == 0.0) return false;
            }
        for (int c = 0; c < 3; ++c) {
            bc->L[c] = box9[4 * c];
            bc->invL[c] = 1.0 / box9[4 * c];
            if (!std::isfinite(bc->invL[c])) return false;
        }
    } else if (box_type == CDH_BOX_TRICLINIC) {
        for (int k = 0; k < 9; ++k) if (!std::isfinite(box9[k])) return false;
        double h_min;
        if (!box_matrices(box9, bc->B, bc->Binv, &h_min)) return false;
        int m = 0;
        for (int i = -1; i <= 1; ++i)
            for (int j = -1; j <= 1; ++j)
                for (int k = -1; k <= 1; ++k, ++m)
                    for (int r = 0; r < 3; ++r)
                        bc->S[m][r] = ((double)i * bc->B[3 * r] + (double)j * bc->B[3 * r + 1]) + (double)k * bc->B[3 * r + 2];
        // pruning: |s_k - n_k| <= 1/2 - 2^-30 is trustworthy while the double error of
        // s_k (<= 15 * 2^-53 * kappa * range, range <= 1024 checked on the device) stays below 2^-31: kappa <= 256.
        double kappa = 0.0;
        for (int k = 0; k < 3; ++k) {
            double row = 0.0;
            for (int c = 0; c < 3; ++c)
                for (int q = 0; q < 3; ++q) row += std::fabs(bc->Binv[3 * k + c]) * std::fabs(bc->B[3 * c + q]);
            kappa = std::fmax(kappa, row);
        }
        bc->prune_ok = (r_max <= 0.5 * h_min * (1.0 + 1e-12) && kappa <= 256.0) ? 1.0 : 0.0;   // slack << the 2^-30 margin
    }
    return true;
}

// Zero structure shared by B and B^-1 (fp32 values): TRI_* of cdh_kernels.cuh.
inline int tri_kind(const BoxConst* bcs, int n) {
    bool upper = true, b01 = true;
    for (int i = 0; i < n; ++i) {
        const float* B = bcs[i].B; const float* Bi = bcs[i].Binv;
        if (B[3] != 0.0f || B[6] != 0.0f || B[7] != 0.0f || Bi[3] != 0.0f || Bi[6] != 0.0f || Bi[7] != 0.0f) upper = false;
        if (B[1] != 0.0f || Bi[1] != 0.0f) b01 = false;
    }
    return !upper ? 0 : (b01 ? 2 : 1);
}

// Bin sweeps ("tiles sized about equal across sweeps").
struct SweepPlan { uint32_t n_sweeps, bins_per_sweep; };
inline SweepPlan plan_sweeps(uint32_t n_bins, uint32_t cap_bins) {
    SweepPlan p;
    p.n_sweeps = (n_bins + cap_bins - 1) / cap_bins;
    p.bins_per_sweep = (n_bins + p.n_sweeps - 1) / p.n_sweeps;
    return p;
}

// Work tables.  Order: histogram row, then sweep, then frame, then i-tile: all items of one (row, sweep)
// key are contiguous, so each CTA flushes O(keys) times.
struct WorkTables {
    std::vector<Seg> segs;
    std::vector<Row> rows;       // + 1 sentinel
    uint64_t n_items = 0;
    uint64_t padded_pairs = 0;   // pair slots the kernel walks (incl. padding and masked lanes)
};

inline void build_tables(int32_t n_frames, const int32_t* off, int32_t n_species, int32_t n_boxes,
                         uint32_t n_bins, const SweepPlan& sp, uint32_t ti, uint32_t tj,
                         const std::vector<uint32_t>& pad_off, uint32_t frame_slots, WorkTables* w) {
    w->segs.clear(); w->rows.clear(); w->n_items = 0; w->padded_pairs = 0;
    uint32_t hist = 0, key = 0;
    for (int p = 0; p < n_species; ++p)
        for (int q = p; q < n_species; ++q, ++hist) {
            const int32_t ni = off[p + 1] - off[p], nj = off[q + 1] - off[q];
            for (uint32_t sw = 0; sw < sp.n_sweeps; ++sw, ++key) {
                if (ni == 0 || nj == 0 || (p == q && ni < 2)) continue;
                const uint32_t lo = sw * sp.bins_per_sweep;
                const uint32_t cnt = (lo + sp.bins_per_sweep <= n_bins) ? sp.bins_per_sweep : n_bins - lo;
                const uint32_t n_jc = ((uint32_t)nj + tj - 1) / tj;
                for (int f = 0; f < n_frames; ++f) {
                    Seg s;
                    s.i_group = (uint32_t)(((uint64_t)f * frame_slots + pad_off[p]) / kGroup);
                    s.j_group = (uint32_t)(((uint64_t)f * frame_slots + pad_off[q]) / kGroup);
                    s.ni = ni; s.nj = nj; s.hist = hist; s.box = (n_boxes == 1) ? 0u : (uint32_t)f;
                    s.same = (p == q); s.bin_lo = lo; s.bin_cnt = cnt; s.key = key;
                    s.last_sweep = (sw + 1 == sp.n_sweeps); s.pad_ = 0;
                    const uint32_t seg_id = (uint32_t)w->segs.size();
                    w->segs.push_back(s);
                    for (uint32_t i0 = 0; i0 < (uint32_t)ni; i0 += ti) {
                        Row r;
                        r.item_prefix = (uint32_t)w->n_items; r.seg = seg_id; r.i0 = i0;
                        r.jc0 = (p == q) ? i0 / tj : 0u;
                        w->rows.push_back(r);
                        w->n_items += n_jc - r.jc0;
                        // the kernel starts at the first 256-particle stage that reaches the diagonal (i0 is a multiple of
                        // the stage) and walks whole j-groups of 4 up to nj
                        w->padded_pairs += (uint64_t)ti * ((((uint32_t)nj + 3u) & ~3u) - ((p == q) ? i0 : 0u));
                    }
                }
            }
        }
    Row sentinel; sentinel.item_prefix = (uint32_t)w->n_items; sentinel.seg = 0; sentinel.i0 = 0; sentinel.jc0 = 0;
    w->rows.push_back(sentinel);
}

}  // namespace cdh
