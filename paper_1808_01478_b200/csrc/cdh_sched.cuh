// cdh_sched.cuh -- K1: the persistent tile kernel (steps S1, S5-S7 of SURVEY.md 8a), generic over the per-pair
// arithmetic.  ONE scheduler for every precision and variant: the arithmetic (steps S2-S4) is a policy class M
// (MathFast / MathSimple in cdh_math32.cuh, MathF64 in cdh_f64.cuh), so the schedule, the stage ring and the flush
// rule cannot drift between the fp32 and the fp64 kernels.
//
// One CTA owns one private uint32 histogram in shared memory (histogram strategy 3, and the
// paper's shared-memory kernel) and works through work items (i-tile, j-chunk): its own index first, then items numbered
// by a global counter, each fetched one item ahead ("Work items" below).
// Items are ordered by (histogram row, bin sweep), so a CTA flushes into the uint64 result only when that key
// changes, when its increment budget nears 2^32 and at exit.  Each thread keeps R = 4
// i-particles in registers; the j-chunk streams through a ring of NS shared-memory stages of 256 particles filled
// by 1-D TMA bulk copies (cp.async.bulk + mbarrier); all lanes read the same j-group (LDS.128 broadcast).
// Intra-species segments only schedule j-chunks that reach above the diagonal (triangular schedule, PAPER.md:137
// Fig. 1, 223-225); stages on the diagonal take the masked form of the arithmetic.
//
// Stage ring: a warp that is done with a stage buffer adds 1 to the buffer's arrival counter; the warp that
// arrives LAST re-arms the buffer's mbarrier and issues the TMA copy of the stage NS ahead into it.  No CTA-wide
// barrier inside a work item: warps drift up to NS - 1 stages apart (with one CTA of 32 warps per SM the
// barrier after every stage of the first version held the warps back for 10 % of their time,
// profiles/r01_cfg5_tile_summary.md "barrier").
#pragma once
#include <type_traits>
#include "cdh_device.cuh"

namespace cdh {

constexpr int kR = 4;                       // i-particles per thread (one group)
constexpr int kSmemHeader = 256;            // 8 mbarriers | spare | 8 arrival counters | two work-item descriptors (64 B each)
constexpr int kMaxStages = 8;
constexpr uint64_t kMaxIncrements = 0xFFFFFFFFull;

// Where the histogram lives: one shared-memory copy of all bins; a shared copy of one bin range per sweep; no private
// copy at all (updates go straight to the uint64 result in L2); a shared window of the bins plus L2 updates for the
// rest, in one sweep (cdh_api.cu "wide histograms").
constexpr int MODE_SHARED = 0, MODE_SPLIT = 1, MODE_GLOBAL = 2, MODE_HYBRID = 3;

// The form of the arithmetic a stage needs: GENERAL drops pairs by the d2 threshold (d >= r_max, NaN padding);
// MASKED also tests j > i (stages on the diagonal of an intra-species segment); CLEAN may assume that every pair of
// the stage is kept (no padding, no NaN coordinate, every distance of the call below r_max -- the policy decides
// per launch whether it can promise that, the scheduler per stage whether the stage holds padding).
constexpr int KIND_GENERAL = 0, KIND_MASKED = 1, KIND_CLEAN = 2;

// What a policy's group() needs to know about the private histogram of the current (row, sweep) key.
struct HistView {
    uint32_t hist_addr;     // shared address of slot 0
    uint32_t trash_addr;    // shared address of the slot that is never flushed
    uint32_t lo, lim;       // first bin and number of slots (bins + the Q3 slot on the last sweep) owned now
    uint32_t last_bin;      // n_bins - 1
    unsigned long long* grow;   // the uint64 result row of the current segment (MODE_GLOBAL / MODE_HYBRID)
};

template <class M>
__host__ __device__ constexpr int tile_smem_fixed(int n_stages) {
    return kSmemHeader + n_stages * M::kStageBytes + (int)((sizeof(typename M::Box) + 15) / 16 * 16) + 16;
}
template <class M>
__host__ __device__ constexpr int tile_smem_bytes(int n_stages, int smem_bins) {
    return tile_smem_fixed<M>(n_stages) + 4 * (smem_bins + 2);     // + Q3 slot + trash slot
}

// SKIP: a warp skips the j-groups that lie below the diagonal for all of its lanes, and every group if it holds only
// padding i-particles (ragged last i-tile).  For frames of small species (a few i-tiles each) this is up to 44 % of a
// diagonal block and half of a ragged tile; the host takes these variants only then (cdh_api.cu), because the
// warp-dependent trip count costs the large-problem kernels 2-5 %.
template <class M, int T, int MINB, int MODE, bool SKIP>
__global__ void __launch_bounds__(T, MINB) tile_kernel(const typename M::Params P) {
    using Real = typename M::Real;
    using Box = typename M::Box;
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int TI = T * kR;
    constexpr uint32_t NW = T / 32;
    constexpr uint32_t kStageBytes = M::kStageBytes;
    constexpr uint32_t kStageReals = kStageGroups * kGroupFloats;
    constexpr uint32_t kGroupBytes = kStageBytes / kStageGroups;
    const uint32_t NS = P.n_stages;                                  // power of two, 2..8
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    uint32_t* s_cons = reinterpret_cast<uint32_t*>(smem + 96);       // [NS] warp arrivals per stage buffer
    ItemDesc* s_slot = reinterpret_cast<ItemDesc*>(smem + 128);      // [2] the work item in hand and the next one (thread 0 fills them)
    unsigned char* stage0 = smem + kSmemHeader;
    Box* s_box = reinterpret_cast<Box*>(smem + kSmemHeader + NS * kStageBytes);
    uint32_t* s_hist = reinterpret_cast<uint32_t*>(smem + tile_smem_fixed<M>((int)NS));
    const uint32_t bar_addr = smem_u32(bars);
    const uint32_t stage_addr = smem_u32(stage0);
    const int tid = threadIdx.x;

    // Work items.  The first item of a CTA is its own index, the later ones are numbered by the global counter.  Thread 0
    // fetches item k + 1 WHILE item k is computed: the counter value it needs was requested one item earlier (the atomic
    // is not waited for until then), and the descriptor travels from the plan's table into the other of two shared-memory
    // slots as an asynchronous copy, so nothing but one CTA barrier stands between two items (the serial chain atomic ->
    // row search -> Row -> Seg of the first version cost configs 2, 4 and 5 2-4 %).  Calls with more items than the table holds
    // look the next item up with ordinary loads at the same point (thread 0's warp then lags by those round trips).
    // A slot whose index field says kNoItem ends the CTA's loop.
    constexpr uint32_t kNoItem = 0xFFFFFFFFu;
    auto fetch_item = [&](const uint32_t item, const uint32_t slot) {
        ItemDesc* dst = s_slot + slot;
        if (item >= P.n_items) { dst->pad_[0] = kNoItem; return; }
        if (P.descs != nullptr) {
            const uint32_t d = smem_u32(dst);
            const unsigned char* q = reinterpret_cast<const unsigned char*>(P.descs + item);
#pragma unroll
            for (int c = 0; c < 4; ++c) cp_async_16(d + 16u * c, q + 16 * c);
        } else {
            uint32_t lo = 0, hi = P.n_rows;         // row of the item: largest r with rows[r].item_prefix <= item
            while (hi - lo > 1) {
                const uint32_t mid = (lo + hi) >> 1;
                if (__ldg(&P.rows[mid].item_prefix) <= item) lo = mid; else hi = mid;
            }
            const Row row = P.rows[lo];
            const uint4* q = reinterpret_cast<const uint4*>(P.segs + row.seg);
            const uint4 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2);
            uint4* o = reinterpret_cast<uint4*>(dst);
            o[0] = a; o[1] = b; o[2] = c;
            o[3] = make_uint4(row.i0, row.jc0 + (item - row.item_prefix), item, 0u);
        }
    };

    // Prologue that reads nothing an earlier kernel of the call writes (the tables are the plan's): it may run while the
    // repack kernel (or the previous tile launch of the call) is still at work (programmatic dependent launch, cdh_api.cu).
    pdl_launch_dependents();
    if (tid == 0) {
        for (uint32_t k = 0; k < NS; ++k) { mbar_init(bar_addr + 8 * k, 1); s_cons[k] = 0; }
        fence_mbar_init();
        fetch_item(blockIdx.x, 0u);
    }
    for (uint32_t b = tid; b <= P.smem_bins + 1; b += T) s_hist[b] = 0;
    pdl_wait();

    // Launch gate: the variants of a call own disjoint intervals of a quantity the repack kernel measured on the
    // device (range of the fractional coordinates for periodic boxes) and exactly one of them does the work; the
    // call never synchronises with the host.  Uniform over the grid.
    typename M::Launch L;
    if (!M::launch_begin(P, L)) return;
    HistView hv;
    hv.hist_addr = smem_u32(s_hist);
    hv.trash_addr = hv.hist_addr + 4u * (P.smem_bins + 1u);          // never flushed
    hv.lo = 0; hv.lim = 0; hv.last_bin = P.n_bins - 1u; hv.grow = P.out;
    const bool one_each = gridDim.x >= P.n_items;      // one CTA per item (small calls): the counter is never touched
    // Claiming an item one item early costs balance at the end of a launch that gives a CTA only a few items (a CTA holds
    // an item it will not start for a while; 10,000 points, 2 items per CTA: 986 Gpairs/s claiming ahead, 1,146 claiming
    // late).  The run-time choice is compiled into the SKIP kernels only -- the ones few-item calls and small species run --
    // because the second code path costs the large-problem kernels 1.0-1.7 % (another ptxas schedule of the pair loops).
    const bool ahead = !SKIP || P.claim_ahead != 0u;
    uint32_t nxt = 0;                                  // thread 0: the counter value that numbers the item to fetch next
    if (tid == 0) {
        if (!one_each && ahead) nxt = atomicAdd(P.counter, 1u);
        cp_async_wait_all();
    }
    __syncthreads();

    uint32_t stage_cnt = 0;                 // stages consumed so far: buffer = cnt % NS, parity = (cnt / NS) & 1
    uint32_t cur_key = 0xFFFFFFFFu, cur_hist = 0, cur_box = 0xFFFFFFFFu;
    uint64_t increments = 0;                // upper bound of increments since the last flush
    const uint32_t ns_mask = NS - 1u, ns_shift = 31u - __clz(NS);

    auto flush = [&]() {
        __syncthreads();
        if (MODE != MODE_GLOBAL && cur_key != 0xFFFFFFFFu) {
            unsigned long long* o = P.out + (size_t)cur_hist * P.n_bins;
            for (uint32_t b = tid; b < hv.lim; b += T) {
                const uint32_t v = s_hist[b];
                if (v) {
                    s_hist[b] = 0;
                    atomicAdd(o + min(hv.lo + b, P.n_bins - 1u), (unsigned long long)v);   // Q3 slot -> last bin
                }
            }
        }
        increments = 0;
        __syncthreads();
    };

    for (uint32_t k = 0;; ++k) {                       // the item in hand is in slot k & 1
        const ItemDesc* d = s_slot + (k & 1u);
        if (d->pad_[0] == kNoItem) break;
        const Seg seg = d->seg;
        const uint32_t i0 = d->i0, jc = d->jc;
        if (tid == 0 && ahead) {
            const uint32_t next_item = one_each ? kNoItem : gridDim.x + nxt;
            fetch_item(next_item, (k + 1u) & 1u);
            if (next_item < P.n_items) nxt = atomicAdd(P.counter, 1u);
        }
        const uint32_t j0 = jc * P.tj;
        const uint32_t j1 = min((uint32_t)seg.nj, j0 + P.tj);

        if (seg.key != cur_key || increments + (uint64_t)TI * P.tj > kMaxIncrements) {
            flush();
            cur_key = seg.key; cur_hist = seg.hist;
            M::template key_begin<MODE>(P, L, seg, hv);              // hv.lo / hv.lim of the new key
        }
        increments += (uint64_t)TI * P.tj;
        hv.grow = P.out + (size_t)seg.hist * P.n_bins;
        if (M::kPeriodic && seg.box != cur_box) {
            __syncthreads();
            const uint32_t* src = reinterpret_cast<const uint32_t*>(P.boxes + seg.box);
            for (int k = tid; k < (int)(sizeof(Box) / 4); k += T) reinterpret_cast<uint32_t*>(s_box)[k] = __ldg(src + k);
            cur_box = seg.box;
            __syncthreads();
        }

        // my R = 4 i-particles (one group) and the constants of the item
        typename M::Item it;
        M::item_begin(P, L, P.pk + ((size_t)seg.i_group + (i0 >> 2) + tid) * kGroupFloats, s_box, hv, it);
        const uint32_t ig = i0 + 4u * tid;          // index of my first i-particle inside the species
        const uint32_t ig_warp = i0 + 4u * ((uint32_t)tid & ~31u);   // first i-particle of my warp (128 consecutive ones)
        const bool warp_idle = ig_warp >= (uint32_t)seg.ni;          // ragged last i-tile: my warp holds padding only
        const bool i_padded = i0 + TI > (uint32_t)seg.ni;            // the i-tile holds NaN padding

        const bool masked = seg.same && (j0 < i0 + TI);       // some j <= some i: test j > i per pair
        const uint32_t n_stage = (j1 - j0 + kStageParticles - 1) / kStageParticles;
        const uint32_t s_begin = (masked && i0 > j0) ? (i0 - j0) / kStageParticles : 0;   // stages wholly below the diagonal
        const Real* jsrc = P.pk + ((size_t)seg.j_group + (j0 >> 2)) * kGroupFloats;

        // fill the ring: the first NS stages of the item (every warp is past the previous item: CTA barrier above)
        if (tid == 0)
            for (uint32_t k = 0; k < NS && s_begin + k < n_stage; ++k) {
                const uint32_t b = (stage_cnt + k) & ns_mask;
                mbar_expect_tx(bar_addr + 8 * b, kStageBytes);
                tma_load_1d(stage_addr + b * kStageBytes, jsrc + (size_t)(s_begin + k) * kStageReals, kStageBytes, bar_addr + 8 * b);
            }
        for (uint32_t s = s_begin; s < n_stage; ++s) {
            const uint32_t b = stage_cnt & ns_mask;
            mbar_wait(bar_addr + 8 * b, (stage_cnt >> ns_shift) & 1u);
            const unsigned char* sj = stage0 + b * kStageBytes;
            const uint32_t jbase = j0 + s * kStageParticles;                   // species index of the stage's first j
            const uint32_t n_left = min(j1 - jbase, (uint32_t)kStageParticles);
            const uint32_t n_grp = (SKIP && warp_idle) ? 0u : (n_left + 3u) >> 2;

            // only stages that touch the diagonal band need the mask; only stages without padding can be CLEAN
            const bool stage_masked = masked && (jbase < i0 + TI);
            auto body = [&](auto kind_c, const uint32_t g_begin) {
                constexpr int KIND = decltype(kind_c)::value;
                // the group's address walks along with g (one add per group; left to itself ptxas rebuilds it from the
                // stage counter in every iteration where registers are short: triclinic kernels, 6 more instructions)
                const unsigned char* pg = sj + g_begin * kGroupBytes;
#pragma unroll M::kUnroll
                for (uint32_t g = g_begin; g < n_grp; ++g, pg += kGroupBytes)
                    M::template group<MODE, KIND, SKIP>(P, L, it, pg, 0u, jbase + 4u * g, ig, hv, s_box);
            };
            if (stage_masked)
                body(std::integral_constant<int, KIND_MASKED>{}, (SKIP && ig_warp > jbase) ? min(n_grp, (ig_warp - jbase) >> 2) : 0u);
            else if (M::kHasClean && L.clean && (M::kCleanPadded || (!i_padded && (n_left & 3u) == 0u && jbase + n_left <= (uint32_t)seg.nj)))
                body(std::integral_constant<int, KIND_CLEAN>{}, 0u);
            else
                body(std::integral_constant<int, KIND_GENERAL>{}, 0u);

            // my warp is done with buffer b; the last warp to say so refills it with the stage NS ahead
            __syncwarp();
            if ((tid & 31) == 0) {
                const uint32_t old = atomicAdd(&s_cons[b], 1u);
                if ((old & (NW - 1u)) == NW - 1u && s + NS < n_stage) {
                    mbar_expect_tx(bar_addr + 8 * b, kStageBytes);
                    tma_load_1d(stage_addr + b * kStageBytes, jsrc + (size_t)(s + NS) * kStageReals, kStageBytes, bar_addr + 8 * b);
                }
            }
            ++stage_cnt;
        }
        if (SKIP && tid == 0 && !ahead)              // claim as late as possible: both round trips are waited for
            fetch_item(one_each ? kNoItem : gridDim.x + atomicAdd(P.counter, 1u), (k + 1u) & 1u);
        if (tid == 0) cp_async_wait_all();
        __syncthreads();              // every warp is done with the item: the ring is reused, the next item is in its slot
    }
    flush();
}

}  // namespace cdh
