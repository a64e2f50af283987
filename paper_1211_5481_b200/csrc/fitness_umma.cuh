// Fused fitness on the 5th-generation tensor cores (scheme GAME_SCHEME_F16X3), sm_100a only.
//
//   z[m,p] = sum_g W[m,g] phi_g(x_p)                      (eq.(2), 61: NP outputs per chromosome)
//   F[m]   = (1/P) sum_p (act(z[m,p]) - t_p)^2            (eq.(3), MSE)
//
// is a dense M x P x G contraction whose B operand (the expansion phi, eq.(1), 79-82 eq.(6)) is
// GENERATED in shared memory and never exists in HBM.  Persistent kernel, one CTA PAIR (cluster of 2, the two
// SMs of a TPC) per 256 chromosomes x 256 patterns tile, tcgen05 cta_group::2:
//
//   warp 0      loader   : cp.async.bulk (1-D TMA) of this CTA's pre-split W operand images, 32 KB (4 K steps) per stage
//   warp 1      MMA      : leader CTA: tcgen05.mma.cta_group::2.kind::f16, M=256 (128 chromosomes per CTA) x
//                          N=256 patterns (128 generated per CTA) x K=16 genes, three MMAs per K step
//                          (W_lo.phi_hi, W_hi.phi_lo, W_hi.phi_hi), fp32 accumulators in TMEM; the whole warp runs the
//                          loop converged and one elected lane issues, so that descriptors stay in uniform registers;
//                          peer CTA: relays "my stage is full" to the leader's barrier
//   warps 2-9   epilogue : tcgen05.ld 32 columns at a time; activation (packed FP32 pairs, one reciprocal per four outputs), (y-t)^2,
//                          private per-chromosome sum (TMEM lane = chromosome, so no shuffle is needed); fp64
//                          accumulation per (CTA, m)
//   warps 10-17 producers: four sets of 2 warps taking pipeline stages in turn; two patterns per thread walking the gene
//                          order with the Chebyshev / multiple-angle recurrences, fp16 hi/lo split, 16-byte stores
//                          straight into the MMA's canonical layout; phi of a pattern tile stays resident in shared
//                          memory and is reused by every chromosome-tile pair of the work unit (see "the kernel")
//
// Why a pair: ncu on the single-CTA version (profiles/r01a) showed the shared-memory data pipe, not the tensor
// pipe, saturating (tensor-core operand reads 46 % + producer stores 28 % + loads 4 % + bulk fills): with
// cta_group::2 each SM reads only its half of B per MMA (8 KB instead of 12 KB) and generates only its 128
// patterns (8 KB of stores per K step instead of 16 KB).
//
// Shared-memory operand layout (both operands): K-major, SWIZZLE_NONE "interleaved" canonical layout with the
// 8-row core matrices packed back to back, i.e. a plain [k_group][row][8 x fp16] array:
//     byte(row, k) = (k / 8) * rows * 16 + row * 16 + (k % 8) * 2        SBO = 128 B, LBO = rows * 16 B
// so a producer warp's 32 rows x 16 B are 512 contiguous bytes (conflict-free) and a K step is any pair of
// k-groups.  The K axis is the gene order of include/game.h without the bias gene (position q = g - 1, 8 positions
// per k-group, zero-padded in the W images to a multiple of 16): no padding inside the K extent, so K steps =
// ceil((G - 1) / 16) (an earlier layout of 8-feature chunks cost c4 9 K steps instead of 8 and c1 6 instead of 4).
// The bias gene a_0 is not on the K axis: the epilogue adds it on the FFMA that scales z for ex2.
#pragma once
#include <cuda_fp16.h>

#include <cstdint>

#include "pdl.cuh"

namespace game {
namespace umma {

constexpr int kBM = 128;             // chromosomes per CTA tile (TMEM lanes); the pair's MMA M is 2 * kBM
constexpr int kBN = 256;             // patterns per pair tile (MMA N, TMEM columns)
constexpr int kRows = kBN / 2;       // pattern rows of the B operand generated and held by each CTA
constexpr int kABytes = 2 * kBM * 16;          // one K step of A, hi or lo: 2 k-groups x 128 rows x 16 B = 4096
constexpr int kBBytes = 2 * kRows * 16;        // one K step of this CTA's half of B, hi or lo: 4096
constexpr int kSlotBytes = 2 * kABytes;        // one K step of either operand (hi + lo) = 8192
static_assert(2 * kBBytes == kSlotBytes, "A and B steps share the slot size");
constexpr int kKS = 4;                         // K steps per pipeline stage: the issuing warp's fixed cost per
                                               // stage (barrier poll, fence, commits) is amortised over 3 * kKS
                                               // MMAs of 128 cycles each (kKS = 1: 27.6 ms, 2: 22.4 ms, 4: 20.3 ms
                                               // per c3 evaluation, measured with a one-lane issue loop)
constexpr int kStageBytes = kKS * kSlotBytes;  // 32768
constexpr int kStagesTotal = 7;                // 32 KB stages shared by the A ring and the B stages (224 KB)
constexpr int kMaxResidentStages = 5;          // phi of a whole pattern tile stays in smem up to 20 K steps
constexpr int kStreamBStages = 3;              // B ring when phi does not fit (regenerated per chromosome tile)
constexpr int kFlushStages = 5;                // streaming mode: the K extent is accumulated in chunks of 5 stages (20 K steps,
                                               // 60 MMAs) and the chunks are added in fp32 by the epilogue.  The tensor core
                                               // adds into the TMEM accumulator with truncation, which shrinks |z| by ~1.6e-8 per
                                               // MMA (measured: 1.25e-5 after the 450 MMAs of G = 2401, identity output); with
                                               // the chunks the shrink is that of one chunk, whatever G is
constexpr int kNumEpiWarps = 8, kNumProdWarps = 8;   // producers: kNumSets sets of kSetWarps warps (128 rows each)
constexpr int kRPT = 2;                        // pattern rows per producer thread: two independent recurrences share one
                                               // walk over the gene order (the walk's control was most of a value's cost)
constexpr int kSetWarps = kRows / (32 * kRPT); // warps that cover the 128 rows of this CTA once: 2
constexpr int kNumSets = kNumProdWarps / kSetWarps;   // producer sets, each takes whole work items: 4
constexpr int kThreads = (2 + kNumEpiWarps + kNumProdWarps) * 32;   // 576
constexpr int kSmemBar = kStagesTotal * kStageBytes;  // barriers start here
constexpr int kAKS = 2;                        // K steps per A ring slot: the A ring is refilled in HALF stages (16 KB), so
                                               // that with two 32 KB stages of A (c3) three refills are in flight while
                                               // one slot is being read; with whole stages the ~1700-cycle refill round
                                               // trip had to fit into one stage's 1536 cycles of tensor time
constexpr int kASlotBytes = kAKS * kSlotBytes; // 16384
constexpr int kMaxASlots = 2 * (kStagesTotal - 1);
constexpr int kBarBytes = (2 * kMaxASlots + 2 * kStagesTotal + 4) * 8 + 16;
constexpr int kTsBytes = kBN * 4;                 // targets of the current pattern tile, staged once per unit
constexpr int kSmemBytes = kSmemBar + kBarBytes + kTsBytes;
constexpr int kTmemCols = 512;                 // two 128 x 256 fp32 accumulators per CTA
constexpr int kStallSlots = 16;                // diagnostic slots per CTA (Params::stall)
#ifndef GAME_EARLY_PRODUCERS
#define GAME_EARLY_PRODUCERS 1
#endif
constexpr bool kEarlyProducers = GAME_EARLY_PRODUCERS != 0;   // the phi producers start before griddepcontrol.wait (A/B switch)
static_assert(kSmemBytes <= 232448, "shared memory budget");
// Operand pre-scaling (both powers of two, so exact, and undone by the epilogue's FFMA constant).  An fp16 hi/lo split is
// only RELATIVE down to 2^-14: below that the lo half is an fp16 subnormal (quantum 2^-24) and an operand of magnitude
// 1e-5 would carry an absolute error of 3e-8.  So each chromosome row is scaled so that its largest gene lands in
// [2^13, 2^14) (a gene 2^15 times smaller than the row's largest still has a normal lo half; below that the absolute
// error is 2^-38 of the row's largest gene), and phi (|phi| <= 1 for Chebyshev on |x| <= 1 and for the trigonometric
// family) is generated times 16 by starting its recurrence from 16 instead of 1 (range: |phi| < 4094).
constexpr int kPhiScaleLog2 = 4;
constexpr float kPhiScale = 16.0f;
constexpr int kRowTargetExp = 13;

struct Params {
    const float* X;        // [P][N]
    const float* t;        // [P]
    const float* W;        // [M][G]: only gene 0 (the bias a_0) is read here, by the epilogue
    const uint8_t* Wimg;   // [m_tiles][steps][8192]: A_hi (2 k-groups x 128 rows x 16 B), then A_lo
    const float* wscale;   // [m_stride]: what the accumulated z of a row has to be multiplied by (row and phi scales undone,
                           //             times the row's calibrated accumulation correction, see calibrate_kernel)
    float* zdump;          // calibration launch only (else NULL): [m_stride][256] raw accumulated z of pattern tile p_tile0;
                           //             no error sums are formed
    double* part;          // [gridDim.x * 2][m_stride] slots of 8 bytes, each holding the running sum as a float-float pair
                           //             (hi, lo): see the epilogue
    const int* stop;       // optional: non-zero => the stop rule is met, the kernel returns at once
    long long* stall;      // optional [gridDim.x][kStallSlots]: cycles the MMA/relay warp waited on a_full, b_full, acc_empty; its total;
                           //          slots 4..: globaltimer stamps of the kernel's phases when built with -DGAME_PROFILE_PHASES
    long long P;
    int N, d, M, G;
    int m_stride;          // m_tiles * 128
    int m_tiles;           // chromosome tiles, padded to an even number (one per CTA of a pair)
    int p_tiles;           // pattern tiles of 256 covered by THIS launch ...
    int p_tile0;           // ... starting at this tile (a generation may be evaluated in several pattern ranges)
    int zero_part;         // 1: this launch starts the generation (clear this CTA's partial sums first)
    int m_groups;          // work unit = (pattern tile, group of m_pairs_per_group chromosome-tile pairs)
    int m_pairs_per_group;
    int dd;                // genes per feature: Chebyshev d, trig 2 d
    int shared;            // 1: the paper's literal model: ONE coefficient set for all features, the term of
                           //    index jj is the SUM over the features; G = dd + 1
    int steps;             // ceil((G - 1) / 16) K steps (the bias gene is added by the epilogue)
    int span;              // K steps per producer work item (kKS; less when the whole K extent is one stage)
    int stages;            // ceil(steps / kKS) pipeline stages per tile
    int resident;          // 1: phi generated once per unit and reused by all its chromosome tiles; n_b == stages, or
                           //    2 * stages (phi of the next unit is generated while this one is consumed)
    int n_a, n_b;          // A ring stages, B stages (n_a + n_b <= kStagesTotal)
    int early;             // 1: the phi producers start their first work item before griddepcontrol.wait (small grids only, see below)
    int flush;             // 1 (streaming mode): accumulate kFlushStages stages at a time, chunk 0 into accumulator 0, the later
                           //    chunks into accumulator 1, which the epilogue adds to accumulator 0 (fp32, round to nearest)
};

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(__cvta_generic_to_shared(p)); }
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same smem offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t local_addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// arrive on a barrier that may live in the other CTA of the pair (address from map_to_cta)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_bar) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Bounded waits: a protocol bug must trap, not hang the GPU.  Default (CTA-scope) semantics on both the remote
// arrive and the wait, as in CUTLASS's ClusterBarrier: cluster-scope acquire/release compile to CCTL.IVALL and
// MEMBAR.ALL.GPU per call, which made the pair kernel 1.7x slower than the single-CTA one.  The data these
// barriers guard is produced for / consumed by the async proxy and is fenced by its writers before they arrive.
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    return done;
}
// The bound of every wait is 20 s of globaltimer, looked at every 2^16 failed polls (a poll count alone could trip under
// time-slicing, MPS or a debugger).
__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void wait_watchdog(uint32_t& n, unsigned long long& t0) {
    if ((++n & 0xffffu) != 0) return;
    const unsigned long long now = global_timer_ns();
    if (t0 == 0) t0 = now;
    else if (now - t0 > 20000000000ull) __trap();
}
// Critical-path waits (MMA issuer, relay, loader): tight poll, three instructions per iteration.
__device__ __forceinline__ void mbar_wait_spin(uint32_t bar, uint32_t parity) {
    uint32_t n = 0;
    unsigned long long t0 = 0;
    while (!mbar_try_wait(bar, parity)) wait_watchdog(n, t0);
}
// Waits of warps that are ahead of the pipeline (producers on a full ring, epilogue on an accumulator still
// being computed): back off with nanosleep so that polling does not steal issue slots from the working warps
// (ncu, profiles/r01a: the clock-checked polling loop was 26 % of all issued warp instructions).
template <int NS>
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity) {
    if (mbar_try_wait(bar, parity)) return;
    uint32_t n = 0;
    unsigned long long t0 = 0;
    do {
        __nanosleep(NS);
        wait_watchdog(n, t0);
    } while (!mbar_try_wait(bar, parity));
}
// The epilogue's accumulator wait: short on the mid-size shapes (the epilogue is the slower side there and a 256 ns nap
// costs ~500 cycles of hand-off), long on the tensor-bound ones (where a spinning warp takes issue slots from the MMA
// warp): poll a few times first, then sleep.
template <int SPINS, int NS>
__device__ __forceinline__ void mbar_wait_spin_then_sleep(uint32_t bar, uint32_t parity) {
#pragma unroll 1
    for (int i = 0; i < SPINS; ++i)
        if (mbar_try_wait(bar, parity)) return;
    uint32_t n = 0;
    unsigned long long t0 = 0;
    do {
        __nanosleep(NS);
        wait_watchdog(n, t0);
    } while (!mbar_try_wait(bar, parity));
}
// Long waits (the producers of a resident unit wait for a whole unit, ~100 us at c3): exponential back-off up to
// MAX_NS.  With a fixed 32 ns sleep this loop was more than half of all instructions the kernel executed (ncu source
// page of a c4 point: 110 M iterations), issue slots and power taken from the working warps.
template <int MAX_NS>
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity) {
    if (mbar_try_wait(bar, parity)) return;
    uint32_t n = 0, ns = 32;
    unsigned long long t0 = 0;
    do {
        __nanosleep(ns);
        ns = min(2 * ns, static_cast<uint32_t>(MAX_NS));
        wait_watchdog(n, t0);
    } while (!mbar_try_wait(bar, parity));
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// TMEM allocation for a CTA pair: issued by the same warp of BOTH CTAs.
__device__ __forceinline__ void tmem_alloc_pair(uint32_t dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t addr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
// One lane of a converged warp (the same lane every time for the same mask).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
// Barrier polls of a converged warp: the elected lane polls, the vote makes the answer warp-uniform.  (All 32 lanes
// polling the same barrier is ruinous when the poll fails: measured 4x on the whole kernel.)
__device__ __forceinline__ bool warp_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
    if (elect_one()) ok = mbar_try_wait(bar, parity);
    return __any_sync(0xffffffffu, ok) != 0;
}
__device__ __forceinline__ void warp_wait_spin(uint32_t bar, uint32_t parity) {
    uint32_t n = 0;
    unsigned long long t0 = 0;
    while (!warp_try_wait(bar, parity)) wait_watchdog(n, t0);
}
// D[tmem, both CTAs] (+)= A[smem of both CTAs] . B[smem of both CTAs]; issued by one thread of the leader CTA.
__device__ __forceinline__ void umma_f16_pair(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// When all MMAs issued so far have completed, arrive once on the barrier at this smem offset in BOTH CTAs.
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
                 "h"(static_cast<unsigned short>(3))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
        "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
        "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]),
        "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]),
        "r"(v[31])
        : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// NaN-propagating clamp (fminf returns the other operand for a NaN, which would turn a NaN z into a finite error).
__device__ __forceinline__ float min_nan(float a, float b) {
    float r;
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}

// Shared-memory matrix descriptor: K-major, SWIZZLE_NONE; start address, LBO (k-group stride) and SBO
// (8-row group stride) in 16-byte units; descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return static_cast<uint64_t>((saddr & 0x3FFFFu) >> 4) | (static_cast<uint64_t>(lbo_bytes >> 4) << 16) |
           (static_cast<uint64_t>(sbo_bytes >> 4) << 32) | (1ull << 46);
}
// The same descriptor in two words: the low one holds the start address (bits 0-13, 16-byte units; shared memory is
// < 256 KB, so adding a byte offset / 16 never carries out of the field) and the k-group stride LBO = 128 rows x 16 B
// (both operands); the high one is constant (SBO = 128 B, descriptor version 1).
static_assert(kBM == kRows, "A and B share the k-group stride");
constexpr uint32_t kDescHiWord = (128u >> 4) | (1u << 14);
constexpr uint32_t kLoHalf = kABytes >> 4;        // hi image -> lo image of the same K step
constexpr uint32_t kNextStep = kSlotBytes >> 4;   // next K step
static_assert(kABytes == kBBytes, "A and B share the image size");
__device__ __forceinline__ uint32_t desc_lo_word(uint32_t saddr) { return ((saddr & 0x3FFFFu) >> 4) | (static_cast<uint32_t>((kBM * 16) >> 4) << 16); }
__device__ __forceinline__ uint64_t desc_from_lo(uint32_t lo) {
    uint64_t d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(kDescHiWord));
    return d;
}
// Instruction descriptor, kind::f16: D = F32 (bit 4), A = B = F16 (0), both K-major, N >> 3 at bit 17,
// M >> 4 at bit 24 (M = 256: the pair's two 128-row halves).
constexpr uint32_t kIdesc = (1u << 4) | (static_cast<uint32_t>(kBN >> 3) << 17) | (static_cast<uint32_t>((2 * kBM) >> 4) << 24);
// ---------------------------------------------------------------------------------------------- K axis
// The K axis is the gene order of include/game.h without the bias gene: position q = g - 1, k-group = 8 consecutive
// positions, K step = 2 k-groups; positions >= G - 1 are padding (zero in the W images, so phi there is irrelevant).
// Gene held by (K step s, k-group kg in {0,1}, slot f in 0..7), or -1 for padding.  Used by the W image builder;
// the producers below generate phi in exactly this order.
__host__ __device__ inline int gene_at(int s, int kg, int f, int G) {
    const int g = 1 + (2 * s + kg) * 8 + f;
    return g < G ? g : -1;
}

// Power-of-two scale of a chromosome row from the largest magnitude among its genes 1..G-1 (the bias gene is not on the K
// axis): 2^k amax in [2^13, 2^14).  Rows without a finite positive maximum (all zero, Inf, NaN) are left unscaled, so
// that non-finite genes still propagate to a non-finite fitness.  k is clamped so that 2^k and 2^-k / 16 stay normal.
__device__ __forceinline__ int row_scale_exp(float amax) {
    if (!(amax > 0.0f) || !(amax < INFINITY)) return 0;
    const int k = kRowTargetExp - ilogbf(amax);
    return max(-100, min(100, k));
}
// The same from the largest |gene| taken as an unsigned integer maximum of the fp32 bit patterns (order-preserving for
// non-negative floats; one redux.sync per warp): a NaN gene has the largest pattern of all and leaves the row unscaled.
__device__ __forceinline__ uint32_t abs_bits(float v) { return __float_as_uint(v) & 0x7fffffffu; }
__device__ __forceinline__ int row_scale_exp_bits(uint32_t amax_bits) { return row_scale_exp(__uint_as_float(amax_bits)); }
// the factor the epilogue applies to the accumulated z of such a row: 2^-k / kPhiScale
__device__ __forceinline__ float row_unscale(int k) { return ldexpf(1.0f, -k - kPhiScaleLog2); }
__device__ __forceinline__ float row_scale_of_unscale(float f) { return 1.0f / (f * kPhiScale); }   // 2^k back from 2^-k / 16: exact

// wscale[m] for every row of the padded population (rows >= M: unscaled).  One warp per row.
__global__ void row_scale_kernel(const float* W, float* wscale, int M, int G, int m_stride) {
    pdl_wait();                // W is complete, and so is the fitness kernel that read the old scales
    pdl_launch_dependents();
    const int m = static_cast<int>((static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (m >= m_stride) return;
    uint32_t amax = 0u;
    if (m < M)
        for (int g = 1 + lane; g < G; g += 32) amax = max(amax, abs_bits(__ldcg(W + static_cast<size_t>(m) * G + g)));
    amax = __reduce_max_sync(0xffffffffu, amax);
    if (lane == 0) wscale[m] = row_unscale(row_scale_exp_bits(amax));
}

// W [M][G] fp32 -> per (m_tile, step) 8 KB images: A_hi then A_lo, each [2 k-groups][128 rows][8 fp16].
// hi = rn_f16(w), lo = rn_f16(w - hi).  One thread per (m_tile, step, k-group, row).
__global__ void build_w_images_kernel(const float* W, const float* wscale, uint8_t* img, int M, int G, int steps, int m_tiles) {
    const long long idx = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    const long long total = static_cast<long long>(m_tiles) * steps * 2 * kBM;
    if (idx >= total) return;
    pdl_wait();                // W and the row scales are complete, and so is the fitness kernel that read the old images
    pdl_launch_dependents();
    const int row = static_cast<int>(idx % kBM);
    const int kg = static_cast<int>((idx / kBM) % 2);
    const int s = static_cast<int>((idx / (2 * kBM)) % steps);
    const int mt = static_cast<int>(idx / (2ll * kBM * steps));
    const int m = mt * kBM + row;
    const float scale = row_scale_of_unscale(__ldcg(wscale + m));
    __half2 hi[4], lo[4];
#pragma unroll
    for (int f2 = 0; f2 < 4; ++f2) {
        float w[2];
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int g = gene_at(s, kg, f2 * 2 + e, G);
            w[e] = (g >= 0 && m < M) ? __ldcg(W + static_cast<size_t>(m) * G + g) * scale : 0.0f;
        }
        const __half2 h = __floats2half2_rn(w[0], w[1]);
        const float2 hf = __half22float2(h);
        hi[f2] = h;
        lo[f2] = __floats2half2_rn(w[0] - hf.x, w[1] - hf.y);
    }
    uint8_t* base = img + (static_cast<size_t>(mt) * steps + s) * (2 * kABytes) + kg * (kBM * 16) + row * 16;
    *reinterpret_cast<uint4*>(base) = *reinterpret_cast<const uint4*>(hi);
    *reinterpret_cast<uint4*>(base + kABytes) = *reinterpret_cast<const uint4*>(lo);
}

// One gene of chromosome m, already multiplied by its row's scale, straight into the W operand images: the same split
// and the same address as build_w_images_kernel, so that the GA step can keep the images of the population it writes up
// to date and the generation loop needs no separate image pass.  Gene 0 (the bias) is not on the K axis.  The zero padding
// (genes past G, rows past M) is written once by build_w_images_kernel and never touched here.
__device__ __forceinline__ void store_w_image_gene(uint8_t* img, int steps, int m, int g, float w) {
    if (g < 1) return;
    const int q = g - 1, kgi = q >> 3, f = q & 7;
    const int s = kgi >> 1, kg = kgi & 1;
    const int mt = m / kBM, row = m % kBM;
    const __half hi = __float2half_rn(w);
    const __half lo = __float2half_rn(w - __half2float(hi));
    uint8_t* base = img + (static_cast<size_t>(mt) * steps + s) * (2 * kABytes) + kg * (kBM * 16) + row * 16 + f * 2;
    *reinterpret_cast<__half*>(base) = hi;
    *reinterpret_cast<__half*>(base + kABytes) = lo;
}

// ---------------------------------------------------------------------------------------------- calibration
// The tensor core adds into its fp32 accumulator with TRUNCATION (round toward zero), so every MMA shrinks |z| a little:
// z_tensor = z (1 - eps), eps ~ 1.6e-8 per MMA (measured: 3.9e-7 for the 24 MMAs of G = 121, 1.25e-5 for the 450 of
// G = 2401).  For a classifier that is far inside the 1e-5 fitness bound, but the error is SYSTEMATIC: on a regression fit
// whose residual r = y - t is small against z it does not average out over the patterns, dF/F = -2 eps <z r> / <r r>,
// up to eps sqrt<z z> / sigma for residual noise sigma (measured 8.9e-5 at sigma = 0.01, identity output).
// So for the regression activations (identity, tanh) the shrink of every chromosome row is MEASURED before each
// evaluation: one extra launch of the fitness kernel hands out the raw accumulators of a sample of <= 256 patterns
// (Params::zdump), cal_phi_kernel + calibrate_kernel recompute the same z for those <= 256 patterns on the CUDA cores (fp32
// expansion as in the producers, products and sums in fp64) and fits z_exact = (1 + eps_m) z_tensor by least squares; the evaluation then runs
// with the row's un-scaling factor times (1 + eps_m).
constexpr int kCalThreads = kBN;         // one thread per sample pattern
constexpr int kCalUnroll = 16;           // K padding of the staged rows

// The sample: n = min(256, rows) patterns spread EVENLY over the knowledge base (rows 0, s, 2 s, ... with s = rows / n),
// copied into a small buffer of the workspace, so that the order of the patterns -- a catalogue sorted by a feature, by
// the target, by anything that correlates with |z| -- does not decide what the fit sees.  (The first 256 patterns as they
// came were the sample until round 3; on a knowledge base sorted by |w* . phi| that left 5e-4 of error on a near-optimal
// identity fit.)  Host-resident knowledge bases are sampled with one strided copy instead (game_api.cu).
__global__ void __launch_bounds__(256) cal_gather_kernel(const float* X, const float* t, float* Xs, float* ts, const int* stop,
                                                         long long n, long long stride, int N) {
    pdl_wait();                // X and t may have been written by whatever ran before on the stream
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; idx < n * N;
         idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long i = idx / N, f = idx - i * N;
        Xs[idx] = __ldcg(X + i * stride * N + f);
    }
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < n; i += static_cast<long long>(gridDim.x) * blockDim.x)
        ts[i] = __ldcg(t + i * stride);
}

// phi of the <= 256 sample patterns, as the producers generate it (fp32 recurrences), widened to
// fp64 once: phi_s[(g - 1) * 256 + p] for genes g = 1..G-1.  One thread per pattern.
template <int EXPANSION>
__global__ void __launch_bounds__(kCalThreads) cal_phi_kernel(const float* __restrict__ X, double* phi_s, const int* stop, long long P,
                                                              int N, int d, int shared) {
    pdl_wait();
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;
    const int p = threadIdx.x;
    const int dd = EXPANSION == 0 ? d : 2 * d;
    const float* xr = X + static_cast<size_t>(p < P ? p : 0) * N;
    if (shared)
        for (int jj = 0; jj < dd; ++jj) phi_s[static_cast<size_t>(jj) * kBN + p] = 0.0;
    // per-feature coefficients: one block per feature; shared coefficients: one block adds up all features (in the
    // producers' order, so that the sums round alike)
    const int i_begin = shared ? 0 : blockIdx.x, i_end = shared ? N : blockIdx.x + 1;
    for (int i = i_begin; i < i_end; ++i) {
        const float x = __ldg(xr + i);
        double* out = phi_s + static_cast<size_t>(shared ? 0 : i * dd) * kBN + p;
        float x2, cm = 1.0f, cc, sm = 0.0f, sc = 0.0f;
        if (EXPANSION == 0) {
            x2 = 2.0f * x; cc = x;
        } else {
            float s1, c1;
            sincosf(x, &s1, &c1);
            x2 = 2.0f * c1; cc = c1; sc = s1;
        }
        for (int k = 0; k < d; ++k) {
            if (shared) {
                out[static_cast<size_t>(k) * kBN] += cc;
                if (EXPANSION == 1) out[static_cast<size_t>(d + k) * kBN] += sc;
            } else {
                out[static_cast<size_t>(k) * kBN] = cc;
                if (EXPANSION == 1) out[static_cast<size_t>(d + k) * kBN] = sc;
            }
            const float cn = fmaf(x2, cc, -cm);
            cm = cc; cc = cn;
            if (EXPANSION == 1) {
                const float sn = fmaf(x2, sc, -sm);
                sm = sc; sc = sn;
            }
        }
    }
}

// zcorr[m] = wscale[m] (1 + eps_m), eps_m from the least-squares fit z_exact = (1 + eps_m) z_tensor over the sample
// patterns.  z_exact = W phi_s is a small fp64 contraction, [M] x [G-1] x [256]: it runs on the fp64 TENSOR path
// (mma.sync m8n8k4 f64), the one fast fp64 unit of this chip -- with scalar DFMA this kernel took 40 us at c2, in
// float-float arithmetic on the FP32 pipe 64 us, against 655 us for the evaluation it calibrates.  A block takes 8
// chromosome rows (genes staged in shared memory as fp64) and all 256 sample patterns, 32 per warp (four 8 x 8 tiles).
constexpr int kCalRows = 8;              // chromosome rows per block = the M of the fp64 MMA
__device__ __forceinline__ void dmma_m8n8k4(double (&acc)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                 : "+d"(acc[0]), "+d"(acc[1])
                 : "d"(a), "d"(b));
}
__global__ void __launch_bounds__(kCalThreads) calibrate_kernel(const float* W, const double* phi_s, const float* zdump,
                                                                const float* wscale, float* zcorr, int* rejected,
                                                                const int* stop, long long P, int M, int G, int m_stride) {
    extern __shared__ double cal_w[];      // [kCalRows][Kp]: the rows' genes 1..G-1 in fp64, zero-padded to a multiple of 16
    __shared__ double s_num[kCalRows][kCalThreads / 32], s_den[kCalRows][kCalThreads / 32];
    pdl_wait();                // the calibration launch's accumulators, phi_s, W and the row scales are complete
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;
    const int m0 = blockIdx.x * kCalRows, tid = threadIdx.x, lane = tid & 31, wv = tid >> 5, K = G - 1;
    const int Kp = (K + 15) / 16 * 16;
    for (int r = 0; r < kCalRows; ++r) {
        const int m = m0 + r;
        for (int g = tid; g < Kp; g += kCalThreads)
            cal_w[static_cast<size_t>(r) * Kp + g] = (m < M && g < K) ? static_cast<double>(__ldcg(W + static_cast<size_t>(m) * G + 1 + g)) : 0.0;
    }
    __syncthreads();
    // fragments of mma.m8n8k4: A (8 x 4, row-major) thread -> (row lane / 4, k lane % 4); B (4 x 8) thread -> (k lane % 4,
    // column lane / 4); C (8 x 8) thread -> row lane / 4, columns 2 (lane % 4) + {0, 1}
    const int fr = lane >> 2, fk = lane & 3;
    double acc[4][2] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    const double* bcol = phi_s + wv * 32 + fr;                     // + k * 256 + 8 j
    const double* arow = cal_w + static_cast<size_t>(fr) * Kp + fk;
    // every block reads the same phi_s: start each block at another K offset, so that they are not all after the same L2
    // lines at the same time (the order of a row's sum still only depends on the row)
    const int k_first = static_cast<int>((static_cast<unsigned>(blockIdx.x) * 16u) % static_cast<unsigned>(Kp));
    for (int it = 0, k0 = k_first; it < Kp; it += 16, k0 = k0 + 16 < Kp ? k0 + 16 : 0) {
        double a[4], b[4][4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {                               // 16 loads of phi in flight per thread
            const int k = k0 + 4 * u + fk;
            a[u] = arow[k0 + 4 * u];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[u][j] = k < K ? __ldcg(bcol + static_cast<size_t>(k) * kBN + 8 * j) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int j = 0; j < 4; ++j) dmma_m8n8k4(acc[j], a[u], b[u][j]);
    }
    // least squares per row over this warp's 32 patterns, then over the warps (fixed order: bit-stable)
    const int n = static_cast<int>(min(static_cast<long long>(kBN), P));
    const int m = m0 + fr;
    double num = 0.0, den = 0.0;
    if (m < m_stride) {
        const double f = static_cast<double>(__ldcg(wscale + m));
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const int p = wv * 32 + 8 * j + 2 * fk + i;
                if (p < n) {
                    const double zt = static_cast<double>(__ldcg(zdump + static_cast<size_t>(m) * kBN + p)) * f;
                    num += (acc[j][i] - zt) * zt;
                    den += zt * zt;
                }
            }
    }
    num += __shfl_xor_sync(0xffffffffu, num, 1); den += __shfl_xor_sync(0xffffffffu, den, 1);
    num += __shfl_xor_sync(0xffffffffu, num, 2); den += __shfl_xor_sync(0xffffffffu, den, 2);
    if (fk == 0) { s_num[fr][wv] = num; s_den[fr][wv] = den; }
    __syncthreads();
    if (tid < kCalRows && m0 + tid < m_stride) {
        const int mm = m0 + tid;
        num = 0.0; den = 0.0;
        for (int w = 0; w < kCalThreads / 32; ++w) { num += s_num[tid][w]; den += s_den[tid][w]; }
        double eps = den == 0.0 ? 0.0 : num / den;      // all-zero outputs: nothing to fit; a NaN / Inf row gives a NaN eps
        // non-finite rows, or a row the model does not describe (the shrink it corrects is ~1e-6): leave it alone, and say so
        // (game_calibration_status counts these rows; one flag per row, written by the row's own thread: no atomics)
        const bool reject = mm < M && !(fabs(eps) <= 1e-4);
        if (rejected != nullptr) rejected[mm] = reject ? 1 : 0;
        if (reject || mm >= M) eps = 0.0;
        zcorr[mm] = static_cast<float>(static_cast<double>(__ldcg(wscale + mm)) * (1.0 + eps));
    }
}

// ---------------------------------------------------------------------------------------------- producer helpers
// lo = v - hi in ONE instruction: the sm_100 mixed-precision FMA (SASS FHFMA) takes the fp16 hi straight from
// the packed register: fma.rn.f32.f16 d = hi * (-1) + v (exact: v - hi is representable).
__device__ __forceinline__ float sub_f16_from_f32(float v, unsigned short hi) {
    float d;
    const unsigned short minus_one = 0xBC00;
    asm("fma.rn.f32.f16 %0, %1, %2, %3;" : "=f"(d) : "h"(hi), "h"(minus_one), "f"(v));
    return d;
}
// Split 8 fp32 values into fp16 hi / lo and store them as one 16-byte k-group row each.
__device__ __forceinline__ void split_store(const float (&v)[8], uint8_t* hi_dst, uint8_t* lo_dst) {
    uint32_t h[4], l[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const __half2 hh = __floats2half2_rn(v[2 * i], v[2 * i + 1]);
        h[i] = *reinterpret_cast<const uint32_t*>(&hh);
        const float l0 = sub_f16_from_f32(v[2 * i], static_cast<unsigned short>(h[i] & 0xffffu));
        const float l1 = sub_f16_from_f32(v[2 * i + 1], static_cast<unsigned short>(h[i] >> 16));
        const __half2 ll = __floats2half2_rn(l0, l1);
        l[i] = *reinterpret_cast<const uint32_t*>(&ll);
    }
    *reinterpret_cast<uint4*>(hi_dst) = make_uint4(h[0], h[1], h[2], h[3]);
    *reinterpret_cast<uint4*>(lo_dst) = make_uint4(l[0], l[1], l[2], l[3]);
}

// (act(z + bias) - t)^2.  `bias_term` is the bias gene pre-multiplied so that it rides on the FFMA that scales z for
// ex2: sigmoid -log2(e) * a_0, tanh 2 log2(e) * a_0, identity a_0 itself.
template <int ACT>
__device__ __forceinline__ float bias_term_of(float a0) {
    return ACT == 1 ? -1.44269504088896340736f * a0 : (ACT == 2 ? 2.88539008177792681472f * a0 : a0);
}
// `tq` is the staged target: t itself, or 1 - t for tanh (so that 1 - 2 r - t is one FFMA).
template <int ACT>
__device__ __forceinline__ float staged_target(float t) { return ACT == 2 ? 1.0f - t : t; }
// `zs` turns the accumulated (pre-scaled) z into the argument: row and phi scales undone, times -log2(e) (sigmoid),
// 2 log2(e) (tanh) or 1 (identity); a power of two times that constant, so no rounding is added.
template <int ACT>
__device__ __forceinline__ float zscale_of(float unscale) {
    return ACT == 1 ? -1.44269504088896340736f * unscale : (ACT == 2 ? 2.88539008177792681472f * unscale : unscale);
}
template <int ACT>
__device__ __forceinline__ float act_err2(float z, float zs, float bias_term, float tq) {
    float e;
    if (ACT == 1) {
        e = rcp_approx(1.0f + ex2_approx(fmaf(z, zs, bias_term))) - tq;
    } else if (ACT == 2) {
        e = fmaf(-2.0f, rcp_approx(1.0f + ex2_approx(fmaf(z, zs, bias_term))), tq);
    } else {
        e = fmaf(z, zs, bias_term) - tq;
    }
    return e * e;
}
// Four outputs at once with ONE reciprocal: r = 1 / (a0 a1 a2 a3), 1 / (a0 a1) = r (a2 a3), 1 / a0 = a1 / (a0 a1), ...
// The epilogue of the mid-size shapes is bound by the MUFU pipe (16 lanes per SM per clock): this is 1.25 MUFU
// operations per output instead of 2 (1.5 with pairs) for 1.25 extra FMULs.  The exponent is clamped at 30 so that the
// product stays finite (<= 2^121); sigmoid / 1 - tanh below 2^-30 are below fp32 resolution of the error against t.
template <int ACT>
__device__ __forceinline__ void act_err2_quad(float z0, float z1, float z2, float z3, float c, float bias_term, float4 tq, float& acc0,
                                              float& acc1, float& acc2, float& acc3) {
    if (ACT == 0) {
        acc0 += act_err2<ACT>(z0, c, bias_term, tq.x);
        acc1 += act_err2<ACT>(z1, c, bias_term, tq.y);
        acc2 += act_err2<ACT>(z2, c, bias_term, tq.z);
        acc3 += act_err2<ACT>(z3, c, bias_term, tq.w);
        return;
    }
    const float a0 = 1.0f + ex2_approx(min_nan(fmaf(z0, c, bias_term), 30.0f));
    const float a1 = 1.0f + ex2_approx(min_nan(fmaf(z1, c, bias_term), 30.0f));
    const float a2 = 1.0f + ex2_approx(min_nan(fmaf(z2, c, bias_term), 30.0f));
    const float a3 = 1.0f + ex2_approx(min_nan(fmaf(z3, c, bias_term), 30.0f));
    const float p01 = a0 * a1, p23 = a2 * a3;
    float r = rcp_approx(p01 * p23);
    if (ACT == 2) r *= -2.0f;                      // tanh = 1 - 2 / a: tq holds 1 - t
    const float r01 = r * p23, r23 = r * p01;      // (-2) / (a0 a1), (-2) / (a2 a3)
    const float s = ACT == 1 ? -1.0f : 1.0f;       // sigmoid: e = 1/a - t; tanh: e = (1 - t) - 2/a
    const float e0 = fmaf(r01, a1, s * tq.x), e1 = fmaf(r01, a0, s * tq.y);
    const float e2 = fmaf(r23, a3, s * tq.z), e3 = fmaf(r23, a2, s * tq.w);
    acc0 = fmaf(e0, e0, acc0);
    acc1 = fmaf(e1, e1, acc1);
    acc2 = fmaf(e2, e2, acc2);
    acc3 = fmaf(e3, e3, acc3);
}

// Packed FP32 pairs (sm_100: FFMA2 / FADD2 / FMUL2 do two IEEE fp32 operations per issued instruction).  The epilogue is
// bound by issue slots and latency, not by the FMA pipe, so halving the FP32 instruction count is what counts.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
// Eight outputs: two interleaved quads (columns 0,2,4,6 and 1,3,5,7), one in each half of the packed operations, each with
// ONE reciprocal per four outputs as in act_err2_quad.  tA, tB: staged targets of columns 0..3 and 4..7.  acc: two packed
// running sums (four scalar sums).
template <int ACT>
__device__ __forceinline__ void act_err2_oct(const uint32_t* v, float c, float bias_term, const float4& tA, const float4& tB, f32x2& acc0,
                                             f32x2& acc1) {
    const f32x2 c2 = pack2(c, c), b2 = pack2(bias_term, bias_term), one2 = pack2(1.0f, 1.0f);
    f32x2 a[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const f32x2 s = fma2(pack2(__uint_as_float(v[2 * k]), __uint_as_float(v[2 * k + 1])), c2, b2);
        float s0, s1;
        unpack2(s, s0, s1);
        // (2^s of part of the pairs from a degree-6 polynomial on the FMA pipe instead of MUFU was measured in rounds 2 and 3
        // and removed: profiles/r03_README.md)
        a[k] = add2(pack2(ex2_approx(min_nan(s0, 30.0f)), ex2_approx(min_nan(s1, 30.0f))), one2);
    }
    const f32x2 p01 = mul2(a[0], a[1]), p23 = mul2(a[2], a[3]);
    float q0, q1;
    unpack2(mul2(p01, p23), q0, q1);
    f32x2 r = pack2(rcp_approx(q0), rcp_approx(q1));
    if (ACT == 2) r = mul2(r, pack2(-2.0f, -2.0f));          // tanh = 1 - 2 / a: the staged target is 1 - t
    const f32x2 r01 = mul2(r, p23), r23 = mul2(r, p01);
    const float sg = ACT == 1 ? -1.0f : 1.0f;                 // sigmoid: e = 1/a - t; tanh: e = (1 - t) - 2/a
    const f32x2 e0 = fma2(r01, a[1], pack2(sg * tA.x, sg * tA.y)), e1 = fma2(r01, a[0], pack2(sg * tA.z, sg * tA.w));
    const f32x2 e2 = fma2(r23, a[3], pack2(sg * tB.x, sg * tB.y)), e3 = fma2(r23, a[2], pack2(sg * tB.z, sg * tB.w));
    acc0 = fma2(e0, e0, acc0);
    acc1 = fma2(e1, e1, acc1);
    acc0 = fma2(e2, e2, acc0);
    acc1 = fma2(e3, e3, acc1);
}

// ---------------------------------------------------------------------------------------------- the kernel
// Shared memory: kStagesTotal stages of 32 KB (kKS = 4 K steps each).  Stages [0, n_a) are the A ring (W operand
// images streamed from L2 by the loader), used as 2 * n_a slots of kAKS = 2 K steps (16 KB); stages
// [n_a, n_a + n_b) hold this CTA's half of B (phi).  If the whole K extent fits (stages <= kMaxResidentStages:
// "resident") phi of a pattern tile is generated ONCE per work unit and reused by every chromosome-tile pair of the
// unit; n_b == stages (the producers refill a stage for the next unit as soon as the unit's last tile has consumed
// it) or, when it fits twice, n_b == 2 * stages (the producers work one unit ahead).  Otherwise ("streaming") B is a
// ring refilled per tile.
//
// Barriers (per CTA unless noted; "leader" = cluster rank 0, "peer" = rank 1):
//   a_full[i]    1 + tx : the loader's bulk copy of A slot i has landed; on the leader +1: the peer's relay
//                         ("my A slot i, and the B stage it pairs with, are full")
//   a_empty[i]   1      : tcgen05.commit of the MMAs that read A slot i, multicast to both CTAs
//   b_full[i]    2 * (K steps in the stage): the 2 producer warps that own each of its K steps have written it
//   b_empty[i]   1      : tcgen05.commit (multicast) of the last MMAs that will read B stage i
//   acc_full[b]  1      : tcgen05.commit after a tile's last MMA, multicast to both CTAs
//   acc_empty[b] 16     : leader only; the 8 epilogue warps of BOTH CTAs have drained accumulator b
struct Ring {
    uint32_t i = 0, phase = 0;
    __device__ __forceinline__ void advance(uint32_t n_stages) {
        if (++i == n_stages) { i = 0; phase ^= 1; }
    }
    __device__ __forceinline__ Ring at(uint32_t offset, uint32_t n_stages) const {
        Ring r = *this;
        r.i += offset;
        while (r.i >= n_stages) { r.i -= n_stages; r.phase ^= 1; }
        return r;
    }
};

template <int EXPANSION, int ACT>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1) fitness_umma_kernel(const Params prm) {
    extern __shared__ __align__(1024) uint8_t smem[];
#ifdef GAME_PROFILE_PHASES
    const unsigned long long ph_entry = global_timer_ns();
#define GAME_PHASE(slot) do { if (prm.stall != nullptr && threadIdx.x == 32) prm.stall[static_cast<size_t>(blockIdx.x) * kStallSlots + (slot)] = static_cast<long long>(global_timer_ns()); } while (0)
#else
#define GAME_PHASE(slot) do { } while (0)
#endif
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kSmemBar);
    const uint32_t bar_a_full = smem_u32(bars), bar_a_empty = bar_a_full + 8 * kMaxASlots;
    const uint32_t bar_b_full = bar_a_empty + 8 * kMaxASlots, bar_b_empty = bar_b_full + 8 * kStagesTotal;
    const uint32_t bar_acc_full = bar_b_empty + 8 * kStagesTotal, bar_acc_empty = bar_acc_full + 16;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * kMaxASlots + 2 * kStagesTotal + 4);
    float* ts_all = reinterpret_cast<float*>(smem + kSmemBar + kBarBytes);
    const uint32_t smem_base = smem_u32(smem);

    // the warp index through a shuffle: ptxas then knows it is warp-uniform, and so is all control flow that depends
    // only on it (the producers' walk over the gene order compiles to uniform branches instead of a convergence
    // barrier per value)
    const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const uint32_t crank = cluster_ctarank();            // 0 = leader, 1 = peer
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    int units = prm.p_tiles * prm.m_groups;
    const int m_pairs = prm.m_tiles >> 1;
    const uint32_t n_a = prm.n_a, n_b = prm.n_b;
    const uint32_t n_as = 2 * n_a;               // A ring slots of kAKS K steps
    const int a_slots = (prm.steps + kAKS - 1) / kAKS;   // A slots per tile
    const int stages = prm.stages;
    const bool resident = prm.resident != 0;
    const uint32_t b_base = smem_base + n_a * kStageBytes;

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kMaxASlots; ++s) {
            mbar_init(bar_a_full + 8 * s, crank == 0 ? 2 : 1);   // leader: own loader + the peer's relay
            mbar_init(bar_a_empty + 8 * s, 1);
        }
        for (int s = 0; s < kStagesTotal; ++s) {
            // K steps held by B stage s (resident: the tile's last stage may hold fewer than kKS)
            const int ks = resident ? min(kKS, prm.steps - (s % stages) * kKS) : kKS;
            mbar_init(bar_b_full + 8 * s, kSetWarps * max(ks, 1));
            mbar_init(bar_b_empty + 8 * s, 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_acc_full + 8 * b, 1);
            mbar_init(bar_acc_empty + 8 * b, 2 * kNumEpiWarps);
        }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc_pair(smem_u32(tmem_slot), kTmemCols);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();          // both CTAs' barriers are initialised before any remote arrive / multicast commit
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
#ifdef GAME_PROFILE_PHASES
    if (prm.stall != nullptr && threadIdx.x == 32) prm.stall[static_cast<size_t>(blockIdx.x) * kStallSlots + 4] = static_cast<long long>(ph_entry);
#endif
    GAME_PHASE(5);             // barriers, TMEM and the cluster handshake done

    // Everything above (barriers, TMEM, the cluster handshake) touches no global memory and overlaps the tail of the
    // preceding kernel (pdl.cuh).  From here on the W images, W, the partial sums and the stop flag are complete.
    // The phi producers do not wait here: all they read is the knowledge base, which no kernel of the chain writes, and all
    // they write is shared memory -- they generate their first work item while the preceding kernel is still running and
    // wait afterwards (late_wait below; every thread of every kernel still passes griddepcontrol.wait before it exits).
    // The host sets Params::early only when the kernel ahead on the stream is one of the library's own (game_api.cu,
    // chain_launches): a caller's kernel that has just rewritten the borrowed X is then at least two launches back and,
    // because every library kernel waits before it releases its dependents, complete.
    // Only for grids that leave SMs free (Params::early): a grid that fills the chip squeezes the GA step it overlaps down to
    // one block per SM, and its busy producers then cost that kernel more than they save here (c1: 48.7 -> 49.6 us per
    // generation; c0, with 8 CTAs, 15.2 -> 13.6 us; the paper-shaped n1 22.5 -> 20.5 us).
    const bool is_producer = kEarlyProducers && prm.early != 0 && warp >= 2 + kNumEpiWarps;
    bool stopped = false;
    if (!is_producer) {
        pdl_wait();
        pdl_launch_dependents();
        GAME_PHASE(6);             // the preceding kernel has completed
        stopped = prm.stop != nullptr && __ldcg(prm.stop) != 0;   // uniform over the grid: written by an earlier kernel
        if (stopped) units = 0;    // stop rule met: no work, no writes; fall through to the teardown (TMEM is allocated)
    }

    if (warp == 0) {
        // ============================================================== loader: W operand images -> A ring
        if (lane == 0) {
            Ring ra;
            uint32_t ready = mbar_try_wait(bar_a_empty + 8 * ra.i, ra.phase ^ 1);
            for (int u = pair; u < units; u += n_pairs) {
                const int mg = u % prm.m_groups;
                const int mp0 = mg * prm.m_pairs_per_group;
                const int mp1 = min(mp0 + prm.m_pairs_per_group, m_pairs);
                for (int mp = mp0; mp < mp1; ++mp) {
                    const int mt = 2 * mp + static_cast<int>(crank);
                    const uint8_t* src = prm.Wimg + static_cast<size_t>(mt) * prm.steps * kSlotBytes;
                    for (int j = 0; j < a_slots; ++j) {
                        if (!ready) mbar_wait_spin(bar_a_empty + 8 * ra.i, ra.phase ^ 1);
                        const uint32_t cur = ra.i;
                        ra.advance(n_as);
                        ready = mbar_try_wait(bar_a_empty + 8 * ra.i, ra.phase ^ 1);   // poll the next slot early
                        const uint32_t bytes = static_cast<uint32_t>(min(kAKS, prm.steps - j * kAKS)) * kSlotBytes;
                        mbar_arrive_expect_tx(bar_a_full + 8 * cur, bytes);
                        bulk_g2s(smem_base + cur * kASlotBytes, src + static_cast<size_t>(j) * kASlotBytes, bytes,
                                 bar_a_full + 8 * cur);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ====================================== MMA issuer (leader) / relay "my stages are full" (peer)
        // The issuing thread is the serial resource of the whole kernel: every instruction between two MMAs shows up
        // in the tile time.  The WHOLE warp runs this loop converged (all lanes poll the barriers) and one elected lane
        // issues the MMAs and commits: everything that feeds them (descriptors, barrier addresses) is then
        // warp-uniform and lives in uniform registers -- under `if (lane == 0)` ptxas wrapped every tcgen05.mma in an
        // elect / 5 x R2UR / branch loop.  A arrives in slots of kAKS K steps (3 * kAKS MMAs per barrier wait); the
        // leader waits on ONE barrier per slot -- its a_full[i] counts its own loader and the peer's relay, and the
        // relay only arrives once the peer's B stage is full too -- and polls the next slot's barrier BEFORE issuing
        // this slot's MMAs.
        Ring ra, rb, rbu;                    // rbu: first B stage of the current unit (resident mode)
        uint32_t tile = 0;
        uint32_t uses0 = 0, uses1 = 0;       // how often each accumulator has been handed to the epilogue so far
        const bool flush = prm.flush != 0;
        const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem_base, 0);
        const uint32_t leader_a_full = map_to_cta(bar_a_full, 0);
        long long st_a = 0, st_b = 0, st_c = 0;
        const long long t_begin = clock64();
        bool ready = warp_try_wait(bar_a_full + 8 * ra.i, ra.phase);
        for (int u = pair; u < units; u += n_pairs, rbu = rbu.at(stages, n_b)) {
            const int mg = u % prm.m_groups;
            const int mp0 = mg * prm.m_pairs_per_group;
            const int mp1 = min(mp0 + prm.m_pairs_per_group, m_pairs);
            for (int mp = mp0; mp < mp1; ++mp, ++tile) {
                const bool need_b = !resident || mp == mp0;          // B stages must be (re)filled for this tile
                const bool release_b = !resident || mp == mp1 - 1;   // last reader of the B stages
                uint32_t buf = 0, d_tmem = 0;
                int k_first = 0;                                      // first K step of the current accumulation chunk
                if (resident) rb = rbu;                               // every tile of the unit reads the same B stages
                for (int j = 0; j < stages; ++j) {
                    if (j == 0 || (flush && j % kFlushStages == 0)) {
                        // a new accumulation: the whole tile (alternating accumulators), or the next chunk of its K extent
                        buf = flush ? (j == 0 ? 0u : 1u) : (tile & 1);
                        d_tmem = tmem_u + buf * kBN;
                        k_first = j * kKS;
                        const uint32_t acc_phase = (buf ? uses1 : uses0) & 1;
                        if (crank == 0 && !warp_try_wait(bar_acc_empty + 8 * buf, acc_phase ^ 1)) {
                            const long long t0 = clock64();
                            warp_wait_spin(bar_acc_empty + 8 * buf, acc_phase ^ 1);
                            st_c += clock64() - t0;
                        }
                        if (buf) ++uses1; else ++uses0;
                    }
                    const bool acc_done = j == stages - 1 || (flush && (j + 1) % kFlushStages == 0);   // this stage ends the accumulation
                    if (need_b && !warp_try_wait(bar_b_full + 8 * rb.i, rb.phase)) {
                        const long long t0 = clock64();
                        warp_wait_spin(bar_b_full + 8 * rb.i, rb.phase);
                        st_b += clock64() - t0;
                    }
                    // the B stage's K steps arrive in A slots of kAKS
                    for (int k0 = j * kKS; k0 < min((j + 1) * kKS, prm.steps); k0 += kAKS) {
                        if (!ready) {
                            const long long t0 = clock64();
                            warp_wait_spin(bar_a_full + 8 * ra.i, ra.phase);
                            st_a += clock64() - t0;
                        }
                        const uint32_t cur = ra.i;
                        ra.advance(n_as);
                        ready = warp_try_wait(bar_a_full + 8 * ra.i, ra.phase);            // next slot's poll, early
                        if (crank == 0) {
                            tc_fence_after();
                            const int k1 = min(k0 + kAKS, prm.steps);
                            const bool last_of_stage = k1 == min((j + 1) * kKS, prm.steps);
                            if (elect_one()) {
                                // The descriptors of a slot differ only in their start-address field (low word, 16-byte units):
                                // one base per operand and constant increments -- lo half + kABytes / 16, next K step +
                                // kSlotBytes / 16.  (Built from scratch per MMA this was 36 instructions per K step in the one
                                // warp whose instruction stream paces the tensor pipe.)
                                const uint32_t a0 = desc_lo_word(smem_base + cur * kASlotBytes);
                                const uint32_t b0 = desc_lo_word(b_base + rb.i * kStageBytes + (k0 - j * kKS) * kSlotBytes);
                                umma_f16_pair(d_tmem, desc_from_lo(a0 + kLoHalf), desc_from_lo(b0), kIdesc, k0 != k_first ? 1u : 0u);   // small terms first
                                umma_f16_pair(d_tmem, desc_from_lo(a0), desc_from_lo(b0 + kLoHalf), kIdesc, 1u);
                                umma_f16_pair(d_tmem, desc_from_lo(a0), desc_from_lo(b0), kIdesc, 1u);
                                if (k1 - k0 > 1) {
                                    static_assert(kAKS == 2, "the issue loop is written out for two K steps per A slot");
                                    const uint32_t a1 = a0 + kNextStep, b1 = b0 + kNextStep;
                                    umma_f16_pair(d_tmem, desc_from_lo(a1 + kLoHalf), desc_from_lo(b1), kIdesc, 1u);
                                    umma_f16_pair(d_tmem, desc_from_lo(a1), desc_from_lo(b1 + kLoHalf), kIdesc, 1u);
                                    umma_f16_pair(d_tmem, desc_from_lo(a1), desc_from_lo(b1), kIdesc, 1u);
                                }
                                umma_commit_pair(bar_a_empty + 8 * cur);                                    // A slot free in both CTAs
                                if (last_of_stage && release_b) umma_commit_pair(bar_b_empty + 8 * rb.i);   // B stage free in both CTAs
                                if (last_of_stage && acc_done) umma_commit_pair(bar_acc_full + 8 * buf);    // accumulation complete
                            }
                            __syncwarp();
                        } else {
                            if (elect_one()) mbar_arrive_cluster(leader_a_full + 8 * cur);      // relay: my slot (and B stage) is full
                            __syncwarp();
                        }
                    }
                    rb.advance(n_b);
                }
            }
        }
        if (prm.stall != nullptr && lane == 0) {
            long long* out = prm.stall + static_cast<size_t>(blockIdx.x) * kStallSlots;
            out[0] = st_a; out[1] = st_b; out[2] = st_c; out[3] = clock64() - t_begin;
        }
    } else if (warp < 2 + kNumEpiWarps) {
        // ============================================================== epilogue
        const int q = warp & 3;                 // TMEM lane quarter this warp may access
        const int h = (warp - 2) >> 2;          // column half
        // The running sum of a (CTA, column half, chromosome) slot is a float-float pair (hi, lo), hi + lo carrying ~48 bits:
        // a tile's fp32 sum is added with an error-free TwoSum (six fp32 adds).  An fp64 add per tile did the same job, but
        // DADD is a slow pipe on this chip (ncu: 6 % of the epilogue warps' samples were that one instruction).
        float2* my_part = reinterpret_cast<float2*>(prm.part) + (static_cast<size_t>(blockIdx.x) * 2 + h) * prm.m_stride;
        if (prm.zero_part && !stopped && prm.zdump == nullptr)
            for (int m = q * 32 + lane; m < prm.m_stride; m += kBM) __stcg(my_part + m, make_float2(0.0f, 0.0f));
        const uint32_t leader_acc_empty = map_to_cta(bar_acc_empty, 0);
        uint32_t tile = 0;
        uint32_t uses0 = 0, uses1 = 0;          // accumulators taken over from the MMA warp so far (barrier phases)
        const bool flush = prm.flush != 0;
        const int n_chunks = flush ? (stages + kFlushStages - 1) / kFlushStages : 1;
        // this thread's target of a unit (column h * 128 + q * 32 + lane of its pattern tile), staged form; 0 if absent
        auto target_of = [&](int uu) {
            if (uu >= units) return 0.0f;
            const long long pp = static_cast<long long>(prm.p_tile0 + uu / prm.m_groups) * kBN + h * 128 + q * 32 + lane;
            return pp < prm.P ? staged_target<ACT>(__ldg(prm.t + pp)) : 0.0f;
        };
        float t_next = target_of(pair);      // always one unit ahead: its HBM latency is hidden behind a whole unit
        // The per-tile scalars of this thread's chromosome row -- bias gene, un-scaling factor, running partial sum -- are
        // fetched ONE TILE AHEAD: loaded at the top of a tile they sat on its critical path (ncu source page of a c4 point:
        // 9 % of the epilogue warps' samples were the first use of the bias, an L2 round trip per tile).
        const bool sums = prm.zdump == nullptr;
        auto row_of = [&](int mp) { return (2 * mp + static_cast<int>(crank)) * kBM + q * 32 + lane; };
        auto first_mp_of = [&](int uu) { return (uu % prm.m_groups) * prm.m_pairs_per_group; };
        int m_nx = pair < units ? row_of(first_mp_of(pair)) : 0;
        float a0_nx = 0.0f, f_nx = 0.0f;          // RAW loaded values: their first use (a multiply) is a tile later
        float2 part_nx = make_float2(0.0f, 0.0f);
        auto fetch_row = [&](int mm) {
            a0_nx = mm < prm.M ? __ldcg(prm.W + static_cast<size_t>(mm) * prm.G) : 0.0f;
            f_nx = __ldcg(prm.wscale + mm);
            if (sums) part_nx = __ldcg(my_part + mm);
        };
        if (pair < units) fetch_row(m_nx);
        for (int u = pair; u < units; u += n_pairs) {
            const int pt = prm.p_tile0 + u / prm.m_groups, mg = u % prm.m_groups;
            const int mp0 = mg * prm.m_pairs_per_group;
            const int mp1 = min(mp0 + prm.m_pairs_per_group, m_pairs);
            const long long p0 = static_cast<long long>(pt) * kBN;
            const int n_valid = static_cast<int>(min(static_cast<long long>(kBN), prm.P - p0));
            // the 4 warps that share a column half stage its 128 targets in shared memory once per unit (they are the
            // same for every chromosome tile of the unit); named barrier per half, 128 threads
            float* ts = ts_all + h * 128;
            asm volatile("bar.sync %0, 128;" ::"r"(2 + h) : "memory");      // everyone is done with the previous tile's t
            ts[q * 32 + lane] = t_next;
            t_next = target_of(u + n_pairs);
            asm volatile("bar.sync %0, 128;" ::"r"(2 + h) : "memory");
            for (int mp = mp0; mp < mp1; ++mp, ++tile) {
                const uint32_t buf = flush ? 0u : (tile & 1);
                const int m = m_nx;
                // the bias gene a_0 is not part of the contraction: it rides on the epilogue's FFMA, together
                // with the row's un-scaling factor; part_old is this lane's running sum
                const float bias = bias_term_of<ACT>(a0_nx), zs = zscale_of<ACT>(f_nx);
                const float2 part_old = part_nx;
                // the next tile's row (of this unit, or the first of this CTA pair's next unit)
                const bool more = mp + 1 < mp1 || u + n_pairs < units;
                m_nx = mp + 1 < mp1 ? row_of(mp + 1) : (u + n_pairs < units ? row_of(first_mp_of(u + n_pairs)) : m);
                const bool same_row = m_nx == m;        // one chromosome tile per unit (M <= 256): carry the sum in the register
                if (more && !same_row) fetch_row(m_nx);
                // streaming mode: accumulator 1 receives the K extent's later chunks one after the other; add each of them to
                // accumulator 0 (chunk 0, then the running sum) with round-to-nearest fp32 adds and hand accumulator 1 back
                for (int chunk = 1; chunk < n_chunks; ++chunk) {
                    mbar_wait_spin_then_sleep<32, 128>(bar_acc_full + 8, uses1 & 1);
                    ++uses1;
                    tc_fence_after();
#pragma unroll 1
                    for (int cc = 0; cc < 4; ++cc) {
                        const int col0 = h * 128 + cc * 32;
                        if (col0 >= n_valid) break;
                        const uint32_t ta = tmem_base + (static_cast<uint32_t>(q * 32) << 16) + col0;
                        uint32_t v0[32], v1[32];
                        tmem_ld32(ta, v0);
                        tmem_ld32(ta + kBN, v1);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i) v0[i] = __float_as_uint(__uint_as_float(v0[i]) + __uint_as_float(v1[i]));
                        tmem_st32(ta, v0);
                    }
                    tmem_st_wait();
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(leader_acc_empty + 8);
                }
                // Short tiles (mid-size shapes): the epilogue is the slower side, the accumulator is usually there already and a
                // nap would only add hand-off time.  Long tiles (tensor-bound shapes): the epilogue idles for most of a tile;
                // sleep through part of that slack first and poll rarely, so that the wait executes next to nothing (polling
                // at the short-tile rate was +1.0 G warp instructions and -4 % tensor-pipe activity at c3 under the power cap).
                mbar_wait_spin_then_sleep<32, 128>(bar_acc_full + 8 * buf, (buf ? uses1 : uses0) & 1);
                if (buf) ++uses1; else ++uses0;
                tc_fence_after();
                float sum = 0.0f, sum1 = 0.0f, sum2 = 0.0f, sum3 = 0.0f;
                f32x2 pacc0 = 0ull, pacc1 = 0ull;      // packed running sums of the full 32-column chunks (sigmoid / tanh)
                // (16 columns at a time with the next chunk's TMEM load in flight was measured twice: 3 % slower.)
#pragma unroll 1
                for (int cc = 0; cc < 4; ++cc) {
                    const int col0 = h * 128 + cc * 32;
                    if (col0 >= n_valid) break;
                    uint32_t v[32];
                    tmem_ld32(tmem_base + (static_cast<uint32_t>(q * 32) << 16) + buf * kBN + col0, v);
                    const float4* tp = reinterpret_cast<const float4*>(ts + cc * 32);
                    tmem_ld_wait();
                    if (prm.zdump != nullptr) {       // calibration launch: hand out the accumulators as they are
                        uint4* zd = reinterpret_cast<uint4*>(prm.zdump + static_cast<size_t>(m) * kBN + col0);
#pragma unroll
                        for (int i = 0; i < 8; ++i) __stcg(zd + i, make_uint4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]));
                        continue;
                    }
                    if (col0 + 32 <= n_valid) {
                        if (ACT == 0) {
#pragma unroll
                            for (int i = 0; i < 8; ++i)
                                act_err2_quad<ACT>(__uint_as_float(v[4 * i + 0]), __uint_as_float(v[4 * i + 1]),
                                                   __uint_as_float(v[4 * i + 2]), __uint_as_float(v[4 * i + 3]), zs, bias, tp[i], sum, sum1,
                                                   sum2, sum3);
                        } else {
#pragma unroll
                            for (int i = 0; i < 4; ++i) act_err2_oct<ACT>(v + 8 * i, zs, bias, tp[2 * i], tp[2 * i + 1], pacc0, pacc1);
                        }
                    } else {
#pragma unroll
                        for (int i = 0; i < 32; ++i) {
                            if (col0 + i < n_valid) sum += act_err2<ACT>(__uint_as_float(v[i]), zs, bias, ts[cc * 32 + i]);
                        }
                    }
                }
                {
                    float p0, p1, p2, p3;
                    unpack2(pacc0, p0, p1);
                    unpack2(pacc1, p2, p3);
                    sum = ((sum + sum1) + (sum2 + sum3)) + ((p0 + p1) + (p2 + p3));
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(leader_acc_empty + 8 * buf);
                if (sums) {
                    const float hi = __fadd_rn(part_old.x, sum);                       // TwoSum: hi + err == part_old.x + sum exactly
                    const float bv = __fadd_rn(hi, -part_old.x);
                    const float err = __fadd_rn(__fadd_rn(part_old.x, -__fadd_rn(hi, -bv)), __fadd_rn(sum, -bv));
                    const float2 part_new = make_float2(hi, __fadd_rn(part_old.y, err));
                    __stcg(my_part + m, part_new);
                    if (same_row) part_nx = part_new;
                }
            }
        }
    } else {
        // ============================================================== producers: phi -> this CTA's half of B
        // Four sets of 2 warps; a thread owns two pattern rows (r and r + 64: two independent recurrences under one walk).
        // A work item is `span` consecutive K steps (one pipeline stage) and the sets take the items in turn.  Within an item a thread walks the flat gene order: it enters the item
        // at feature i, index j within the feature (re-running the recurrence up to j), emits 8 values per k-group and
        // moves to the next feature whenever j reaches dd; all of this control is uniform over the warp.  x is read
        // straight from global memory in blocks of four features, one block ahead (the rows of the NEXT unit are prefetched
        // into L2 meanwhile).  One proxy fence + the arrivals per item.
        const int pw = warp - (2 + kNumEpiWarps);       // producer warp 0..7
        const int set = pw / kSetWarps;                  // which warp set
        const int r = (pw % kSetWarps) * 32 + lane;      // first pattern row of this thread; it also owns r + 64
        const int dd = prm.dd, span = prm.span;
        const int n_items = (prm.steps + span - 1) / span;
        Ring rb;                                // ring position of the current fill's first stage
        uint32_t item = 0;                      // running item counter: item goes to set (item & 1)
        // griddepcontrol.wait, late: after this thread's first work item, or before its second unit, or on the way out.
        // Only then is the stop flag of game_run_until known: a stopped launch has filled at most one stage for nobody,
        // which the teardown does not mind.
        bool waited = false;
        auto late_wait = [&]() {
            if (waited) return;
            waited = true;
            pdl_wait();
            pdl_launch_dependents();
            if (prm.stop != nullptr && __ldcg(prm.stop) != 0) units = 0;
        };
        for (int u = pair; u < units; u += n_pairs) {
            if (u != pair) {
                late_wait();
                if (units == 0) break;
            }
            const int pt = prm.p_tile0 + u / prm.m_groups, mg = u % prm.m_groups;
            const int mp0 = mg * prm.m_pairs_per_group;
            const int mp1 = min(mp0 + prm.m_pairs_per_group, m_pairs);
            // x in blocks of 4 features.  Block b of a row; b and the feature indices are clamped into the row, so a
            // load never leaves it (features past N only exist in the zero-padded tail of the K axis, where phi is
            // multiplied by W image zeros: any finite value of the SAME row will do there, and a row that holds a
            // non-finite value has a non-finite z anyway).  Rows of a pattern past P read the launch's first row (masked by the
            // epilogue; with an out-of-core knowledge base only this launch's pattern range is in device memory).
            const float* xrow[kRPT];
#pragma unroll
            for (int q = 0; q < kRPT; ++q) {
                const long long p = static_cast<long long>(pt) * kBN + static_cast<long long>(crank) * kRows + r + q * (kRows / kRPT);
                xrow[q] = prm.X + (p < prm.P ? p : static_cast<long long>(prm.p_tile0) * kBN) * prm.N;
            }
            const bool vec4 = (prm.N & 3) == 0;       // rows are 16-byte aligned (X itself is: game_load_kb checks)
            const int last_blk = (prm.N - 1) >> 2, last_i = prm.N - 1;
            auto fetch4 = [&](const float* row, int b) {
                b = min(b, last_blk);
                if (vec4) return __ldg(reinterpret_cast<const float4*>(row) + b);
                const int i0 = 4 * b;
                return make_float4(__ldg(row + i0), __ldg(row + min(i0 + 1, last_i)), __ldg(row + min(i0 + 2, last_i)),
                                   __ldg(row + min(i0 + 3, last_i)));
            };
            // the knowledge base streams from HBM exactly once: pull the next unit's rows into L2 now, so that its first
            // loads do not pay the HBM latency on the critical path of a short unit
            if (set == 0 && u + n_pairs < units) {
#pragma unroll
                for (int q = 0; q < kRPT; ++q) {
                    const long long pn = static_cast<long long>(prm.p_tile0 + (u + n_pairs) / prm.m_groups) * kBN +
                                         static_cast<long long>(crank) * kRows + r + q * (kRows / kRPT);
                    if (pn < prm.P) {
                        const char* row = reinterpret_cast<const char*>(prm.X + pn * prm.N);
                        const int bytes = prm.N * 4;
                        for (int off = 0; off < bytes; off += 128) prefetch_l2(row + off);
                        prefetch_l2(row + bytes - 4);
                    }
                }
            }
            const int n_fill = resident ? 1 : mp1 - mp0;        // how many times the K extent is generated
            for (int fill = 0; fill < n_fill; ++fill) {
                for (int w = 0; w < n_items; ++w, ++item) {
                    const int s0 = w * span, s1 = min(prm.steps, s0 + span);
                    const Ring pos = rb.at(s0 / kKS, n_b);
                    if (item % kNumSets != static_cast<uint32_t>(set)) {
                        // Not this set's item, but still wait for its stage to have been emptied: an mbarrier wait only
                        // tells one phase from the next, so a set must watch EVERY lap of every stage go by (with more
                        // sets than ring stages it would otherwise skip a lap and take a stale phase for the one it
                        // needs).  Stages are released in item order, so this never delays the set's own item.
                        mbar_wait_backoff<512>(bar_b_empty + 8 * pos.i, pos.phase ^ 1);
                        continue;
                    }
                    if (prm.shared) {
                        // ---- shared coefficients: term jj of a pattern = sum over its features of T_{jj+1}(x_i) (or cos / sin).
                        // One k-group (8 consecutive jj) at a time: for every feature the recurrence is run from its start
                        // up to the k-group and the 8 values are added up; the K extent is short (dd <= 64), so re-running
                        // the head of the recurrence costs less than keeping dd accumulators per row would.
                        mbar_wait_backoff<512>(bar_b_empty + 8 * pos.i, pos.phase ^ 1);
                        uint8_t* dst = smem + (n_a + pos.i) * kStageBytes + (s0 % kKS) * kSlotBytes + r * 16;
#pragma unroll 1
                        for (int g8 = 0; g8 < 2 * (s1 - s0); ++g8) {
                            const int jbase = 8 * (2 * s0 + g8);
                            float acc[kRPT][8];
#pragma unroll
                            for (int q = 0; q < kRPT; ++q)
#pragma unroll
                                for (int e = 0; e < 8; ++e) acc[q][e] = 0.0f;
                            float4 blk[kRPT];
#pragma unroll 1
                            for (int i = 0; i < prm.N; ++i) {
                                float x2[kRPT], cp[kRPT], cc[kRPT], sp[kRPT], sc[kRPT];
#pragma unroll
                                for (int q = 0; q < kRPT; ++q) {
                                    if ((i & 3) == 0) blk[q] = fetch4(xrow[q], i >> 2);
                                    const int k = i & 3;
                                    const float x = k == 0 ? blk[q].x : (k == 1 ? blk[q].y : (k == 2 ? blk[q].z : blk[q].w));
                                    if (EXPANSION == 0) {      // the recurrences are linear: started from kPhiScale they yield kPhiScale * phi
                                        x2[q] = 2.0f * x; cp[q] = kPhiScale; cc[q] = kPhiScale * x; sp[q] = 0.0f; sc[q] = 0.0f;
                                    } else {
                                        float sn, cs;
                                        sincosf(x, &sn, &cs);
                                        x2[q] = 2.0f * cs; cp[q] = kPhiScale; cc[q] = kPhiScale * cs; sp[q] = 0.0f; sc[q] = kPhiScale * sn;
                                    }
                                }
                                auto step = [&](int q, int jj) {
                                    float out;
                                    if (EXPANSION == 0 || jj < prm.d) {
                                        out = cc[q];
                                        const float t = fmaf(x2[q], cc[q], -cp[q]);
                                        cp[q] = cc[q]; cc[q] = t;
                                    } else {
                                        out = sc[q];
                                        const float t = fmaf(x2[q], sc[q], -sp[q]);
                                        sp[q] = sc[q]; sc[q] = t;
                                    }
                                    return out;
                                };
                                for (int jj = 0; jj < jbase; ++jj) {
#pragma unroll
                                    for (int q = 0; q < kRPT; ++q) step(q, jj);
                                }
#pragma unroll
                                for (int e = 0; e < 8; ++e) {
#pragma unroll
                                    for (int q = 0; q < kRPT; ++q) acc[q][e] += step(q, jbase + e);
                                }
                            }
#pragma unroll
                            for (int q = 0; q < kRPT; ++q)
                                split_store(acc[q], dst + q * (kRows / kRPT) * 16, dst + q * (kRows / kRPT) * 16 + kBBytes);
                            dst += (g8 & 1) ? kRows * 16 + kBBytes : kRows * 16;
                        }
                    } else {
                    // where this item enters the gene order
                    int i = (16 * s0) / dd, j = 16 * s0 - i * dd;
                    // x in blocks of 4 features (one 16-byte load per block when the rows are 16-byte aligned: a scalar
                    // load of one feature touches 32 different lines per warp, and those loads were what bounded the
                    // producers on short units); `cur` is the block of feature i, `nxt` the one after it, already in flight
                    float4 cur[kRPT], nxt[kRPT];
#pragma unroll
                    for (int q = 0; q < kRPT; ++q) {
                        cur[q] = fetch4(xrow[q], i >> 2);
                        nxt[q] = fetch4(xrow[q], (i >> 2) + 1);
                    }
                    auto pick = [&](const float4& c4, int ii) {
                        const int k = ii & 3;
                        return k == 0 ? c4.x : (k == 1 ? c4.y : (k == 2 ? c4.z : c4.w));
                    };
                    // recurrence state per row: cp, cc = T_j, T_{j+1} (or cos jx, cos (j+1)x); sp, sc = sin jx, sin (j+1)x
                    float x2[kRPT], cp[kRPT], cc[kRPT], sp[kRPT], sc[kRPT];
                    auto enter = [&]() {                      // both rows start feature i
#pragma unroll
                        for (int q = 0; q < kRPT; ++q) {
                            const float x = pick(cur[q], i);
                            if (EXPANSION == 0) {      // started from kPhiScale the (linear) recurrences yield kPhiScale * phi
                                x2[q] = 2.0f * x; cp[q] = kPhiScale; cc[q] = kPhiScale * x; sp[q] = 0.0f; sc[q] = 0.0f;
                            } else {
                                float sn, cs;
                                sincosf(x, &sn, &cs);
                                x2[q] = 2.0f * cs; cp[q] = kPhiScale; cc[q] = kPhiScale * cs; sp[q] = 0.0f; sc[q] = kPhiScale * sn;
                            }
                        }
                    };
                    // value of index jj within the feature (Chebyshev T_{jj+1}; trig cos (jj+1)x for jj < d, else
                    // sin (jj-d+1)x) of row q, advancing the recurrence that produced it
                    auto next = [&](int q, int jj) {
                        float out;
                        if (EXPANSION == 0 || jj < prm.d) {
                            out = cc[q];
                            const float t = fmaf(x2[q], cc[q], -cp[q]);
                            cp[q] = cc[q]; cc[q] = t;
                        } else {
                            out = sc[q];
                            const float t = fmaf(x2[q], sc[q], -sp[q]);
                            sp[q] = sc[q]; sc[q] = t;
                        }
                        return out;
                    };
                    enter();
                    for (int jj = (EXPANSION == 0 || j <= prm.d) ? 0 : prm.d; jj < j; ++jj) {
#pragma unroll
                        for (int q = 0; q < kRPT; ++q) next(q, jj);
                    }
                    mbar_wait_backoff<512>(bar_b_empty + 8 * pos.i, pos.phase ^ 1);
                    // One k-group (8 values, one 16-byte row of hi and of lo, for each of the thread's rows) per iteration
                    // of a loop that is NOT unrolled: unrolled over the 16 values of a K step the body was 25 KB of code, a
                    // quarter of the producers' stall samples were instruction-cache misses (ncu source page of an M = 256
                    // point) and 21 warp instructions were executed per value.  (A one-value-per-iteration loop with a
                    // sliding 8-value window was smaller still, but its serial chain made an item 25 % slower.)
                    uint8_t* dst = smem + (n_a + pos.i) * kStageBytes + (s0 % kKS) * kSlotBytes + r * 16;
#pragma unroll 1
                    for (int g8 = 0; g8 < 2 * (s1 - s0); ++g8) {
                        float v[kRPT][8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            if (j == dd) {
                                ++i; j = 0;
                                if ((i & 3) == 0) {
#pragma unroll
                                    for (int q = 0; q < kRPT; ++q) { cur[q] = nxt[q]; nxt[q] = fetch4(xrow[q], (i >> 2) + 1); }
                                }
                                enter();
                            }
#pragma unroll
                            for (int q = 0; q < kRPT; ++q) v[q][e] = next(q, j);
                            ++j;
                        }
#pragma unroll
                        for (int q = 0; q < kRPT; ++q)
                            split_store(v[q], dst + q * (kRows / kRPT) * 16, dst + q * (kRows / kRPT) * 16 + kBBytes);
                        dst += (g8 & 1) ? kRows * 16 + kBBytes : kRows * 16;   // next k-group; after the odd one skip the lo half
                    }
                    }   // per-feature coefficients
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) {
                        for (int st = s0; st < s1; ++st) {
                            mbar_arrive(bar_b_full + 8 * pos.i);
                            // streaming ring stages always expect kKS K steps: stand in for the missing ones
                            if (!resident && st == prm.steps - 1)
                                for (int e = prm.steps % kKS; e != 0 && e < kKS; ++e) mbar_arrive(bar_b_full + 8 * pos.i);
                        }
                    }
                    late_wait();
                    if (units == 0) break;
                }
                if (units == 0) break;
                rb = rb.at(stages, n_b);
            }
        }
        late_wait();
    }

    GAME_PHASE(7);             // the MMA warp has issued everything
    // ---- teardown: everything issued has been consumed once both epilogues have drained the last accumulator;
    // neither CTA may exit (or free TMEM) while the other can still signal its barriers or read its operands.
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();
    tc_fence_after();
    GAME_PHASE(8);             // both CTAs are through
    if (warp == 1) {
        __syncwarp();
        tmem_dealloc_pair(tmem_base, kTmemCols);
    }
    GAME_PHASE(9);
#undef GAME_PHASE
}

}  // namespace umma
}  // namespace game
