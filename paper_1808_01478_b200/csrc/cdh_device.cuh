// cdh_device.cuh -- device-side data structures and small PTX helpers of libcdh (sm_100a only).
//
// Everything here is independent of the CPU oracle under oracle/ (no shared code, headers or tables).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cdh {

// ---------------------------------------------------------------------------------------------
// Layout of the repacked coordinates (step S0; "pad triple to 4"):
// groups of 4 particles, 12 floats per group: x0 x1 x2 x3 | y0 y1 y2 y3 | z0 z1 z2 z3 (48 bytes, no
// padding bytes).  Each species of each frame starts on a group boundary and is padded with NaN up to
// a multiple of kPadParticles particles, so a thread's register tile and a TMA stage never read out of
// bounds and padding lanes drop out of the histogram by the same d2 test that drops NaN inputs.
// ---------------------------------------------------------------------------------------------
constexpr int kGroup = 4;                 // particles per group
constexpr int kGroupFloats = 12;          // floats per group
#ifndef CDH_STAGE
#define CDH_STAGE 256   // measured: 256 vs 512 gives cfg2 +1.7 % (finer work items, shorter tail), 128 no further gain
#endif
constexpr int kStageParticles = CDH_STAGE; // j-particles per shared-memory stage (3 KB in fp32, 6 KB in fp64)
constexpr int kStageGroups = kStageParticles / kGroup;
constexpr int kStageBytes = kStageGroups * kGroupFloats * 4;
#ifndef CDH_PAD
#define CDH_PAD 4096
#endif
constexpr int kPadParticles = CDH_PAD;    // multiple of every i-tile size (threads * 4) and of kStageParticles

// One (frame, species pair, bin sweep).  Work items of a segment are (i-tile, j-chunk) pairs.
struct Seg {
    uint32_t i_group;   // first group of species p of this frame in the repacked buffer
    uint32_t j_group;   // first group of species q
    int32_t  ni, nj;    // particles in p and q
    uint32_t hist;      // output row
    uint32_t box;       // index into the box-constant table
    uint32_t same;      // 1: p == q, count only j > i
    uint32_t bin_lo;    // first bin owned by this sweep
    uint32_t bin_cnt;   // bins owned by this sweep
    uint32_t key;       // (hist, sweep) id: a CTA flushes its private histogram when the key changes
    uint32_t last_sweep;// 1: the sweep that owns bin n_bins-1 (and the Q3 overflow slot)
    uint32_t pad_;
};

// One i-tile of one segment: its items are the j-chunks jc0 .. n_jc-1.
struct Row {
    uint32_t item_prefix;  // index of the row's first item in the global item order
    uint32_t seg;
    uint32_t i0;           // first particle of the i-tile inside species p (multiple of the tile size)
    uint32_t jc0;          // first j-chunk
};

// Per-box constants in fp32, derived on the host in double and rounded once (DESIGN.md
// "Host-derived constants").  B has the box vectors as COLUMNS (Eq. 5).
struct BoxConst {
    float S[27][4];             // TRICLINIC: shift vectors ((i*B[r][0] + j*B[r][1]) + k*B[r][2]), i,j,k in -1..1; [3] = 0
                                // (first member: 16-byte aligned in shared memory, one LDS.128 per shift)
    float L[3], invL[3];        // ORTHO
    float invLf[3];             // ORTHO_FUSED: the constant of the fused rint (host search, fused_rint_constant)
    float B[9], Binv[9];        // TRICLINIC, row-major
    float prune_ok;             // TRICLINIC 1: r_max <= h_min/2 with margin, the zero-shift candidate may be tested alone
                                // ORTHO 1: fused rint constants exist for all three axes
};
static_assert(sizeof(BoxConst) % 16 == 0, "BoxConst is copied and indexed in 16-byte units");

// Everything the scheduler needs to know about one work item, so that a CTA learns it in one (asynchronous) copy instead
// of four dependent round trips to memory (row search, Row, Seg).  Built by the host unless the call has very many items.
struct alignas(16) ItemDesc {
    Seg seg;
    uint32_t i0, jc;            // first particle of the i-tile inside species p, j-chunk
    uint32_t pad_[2];           // [0]: the item's index (0xFFFFFFFF in a shared-memory slot: no item left)
};
static_assert(sizeof(Seg) == 48 && sizeof(ItemDesc) == 64, "ItemDesc is copied as four 16-byte words");

// The part of the tile kernel's parameters that does not depend on the precision (cdh_sched.cuh).
struct TileCommon {
    const Seg*      segs;
    const Row*      rows;       // n_rows + 1 entries (last: item_prefix = n_items)
    const ItemDesc* descs;      // n_items entries, or nullptr (calls with very many items look the item up in rows / segs)
    unsigned int*   counter;    // dynamic work counter of the items past the first one of every CTA (zero before the launch)
    unsigned long long* out;    // uint64 [n_hist][n_bins]
    const unsigned int* range_keys;  // device, written by the repack kernel: [0..2] max keys, [3..5] complemented min keys of the
                                     // fractional coordinates (periodic boxes) or of the raw coordinates (no box), [6] != 0: some
                                     // particle has a NaN coordinate
    const uint32_t* win_lo;     // MODE_HYBRID: first bin of the shared-memory window of each histogram row (device; window_kernel)
    uint32_t n_rows, n_items;
    uint32_t n_bins;
    uint32_t tj;                // j-chunk size in particles (a multiple of kStageParticles, or 32 / 64 / 128 for small calls)
    uint32_t smem_bins;         // capacity of the shared histogram (bins per sweep / window, without the two extra slots)
    uint32_t n_stages;          // stages of the TMA ring (power of two, 2..8)
    uint32_t claim_ahead;       // SKIP kernels: 1 = a CTA claims its next work item one item early (launches with >= 16 items per CTA)
};

struct TileParams : TileCommon {
    const float*    pk;         // repacked coordinates
    const BoxConst* boxes;
    float rmax, scale;          // (float)r_max, (float)(n_bins / r_max)
    uint32_t thr2_bits;         // bits of the smallest fp32 d2 whose correctly rounded sqrt is >= rmax
    float one;                  // 1.0f, opaque to ptxas: keeps packed mul/add pairs unfused
    float one_u;                // 1.0f once more, for FFMA2 whose other two operands are register pairs: ptxas keeps this copy
                                // in a uniform register (the first one must be a vector register where the addend is an immediate)
    float range_lo, range_hi;   // periodic boxes: this launch does the work iff range_lo < frac_range() <= range_hi
                                // (range_hi = +inf: no upper limit, and a NaN range counts as above range_lo)
    uint32_t keep_bins;         // 0, or (orthorhombic box, this launch only) the number of flushed slots of a private histogram that
                                // has a slot for EVERY reachable distance: stages without padding then need no threshold compare
                                // (DESIGN.md "CLEAN form"); smem_bins is the full slot count
};

// ---------------------------------------------------------------------------------------------
// PTX helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// Programmatic dependent launch (cdh_api.cu launches the tile kernels with programmatic stream serialization): a kernel
// lets the next one in the stream start its prologue early, and the next one waits here -- for the COMPLETION of every
// kernel before it -- before it touches anything an earlier kernel of the stream writes.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// 16-byte asynchronous copy global -> shared (LDGSTS) and the wait for all copies of the executing thread
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// 1-D TMA bulk copy global -> shared, completion on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// Shared-memory histogram increment, no return value (SASS: ATOMS.POPC.INC / ATOMS.ADD with RZ dest).
__device__ __forceinline__ void hist_inc(uint32_t addr) {
    asm volatile("red.shared.add.u32 [%0], 1;" ::"r"(addr) : "memory");
}
// Predicated form: a single @P ATOMS instead of a branch around the atomic.
__device__ __forceinline__ void hist_inc_if(bool keep, uint32_t addr) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %1, 0;\n@p red.shared.add.u32 [%0], 1;\n}\n" ::"r"(addr), "r"((uint32_t)keep) : "memory");
}
// Global uint64 counter += 1 under a predicate, no return value (SASS: @P REDG.E.ADD.64): no branch around the reduction.
__device__ __forceinline__ void red_global_inc_if(bool keep, unsigned long long* addr) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %1, 0;\n@p red.global.add.u64 [%0], 1;\n}\n" ::"l"(addr), "r"((uint32_t)keep) : "memory");
}
__device__ __forceinline__ void hist_add(uint32_t addr, uint32_t v) {
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// Packed f32x2 arithmetic (sm_100: FADD2 / FMUL2 / FFMA2; IEEE round-to-nearest-even per element).
typedef unsigned long long f2;   // two floats in one 64-bit register pair: lo = element 0
__device__ __forceinline__ f2 pk2(float a, float b) {
    f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r;
}
__device__ __forceinline__ void upk2(f2 v, float& a, float& b) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ f2 sub2(f2 a, f2 b) {
    f2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b) {
    f2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 add2_rm(f2 a, f2 b) {   // round toward -inf
    f2 r; asm("add.rm.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b) {
    f2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) {
    f2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
}
__device__ __forceinline__ f2 fma2_rm(f2 a, f2 b, f2 c) {   // round toward -inf
    f2 r; asm("fma.rm.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
}

}  // namespace cdh
