// GA operators on the device: population init, one whole generation in ONE kernel, and the fixed-order
// fitness finalisation.  PAPER.md:43 names the operators (crossover, mutation, selection, elitism) and
// PAPER.md:134-136 their rates; their definitions are the readings of SURVEY 8(c) R6-R8 / DESIGN.md
// (tournament with replacement, single-point crossover, per-gene Gaussian mutation, BASELINE.json).
// PAPER.md:170 lists moving "population formation and evolution" to the GPU as future work (i): this is it.
#pragma once
#include <cmath>
#include <cstdint>

#include "fitness_umma.cuh"
#include "pdl.cuh"
#include "philox.cuh"

namespace game {

constexpr int kGaThreads = 128;

// ---- order on chromosomes (R7.1): a precedes b iff key(F[a]) < key(F[b]), ties -> lower index;
// key(NaN) = +inf (NaN fitness is worst).  Lower fitness (MSE) is better (D4).
__device__ __forceinline__ float fit_key(float f) { return (f != f) ? INFINITY : f; }
// The error a fitness value stands for.  MSE / RMSE are errors themselves; under the paper's literal fitness 1 - error,
// maximised (GAME_ERROR_ONE_MINUS_MSE) the operators work on e = 1 - fitness (one fp32 subtraction, exact for
// fitness in [1/2, 1]), so that every operator is the SAME function of an error vector whatever is reported.  What is NOT
// exact is the rounding of 1 - MSE to fp32 when the fitness was written (spacing 6e-8 below 1): errors closer than that tie.
// include/game.h (game_set_error_metric, "RESOLUTION") says when to search on the MSE itself instead.
__device__ __forceinline__ float err_view(float f, int maximize) { return maximize ? 1.0f - f : f; }

__device__ __forceinline__ bool precedes(float ka, int a, float kb, int b) {
    return (ka < kb) || (ka == kb && a < b);
}

// ---- population init (R6): one thread per Philox block = 4 consecutive genes.
__global__ void init_population_kernel(float* __restrict__ W, int M, int G, PhiloxKey key) {
    const int groups = (G + 3) >> 2;
    const long long idx = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (idx >= static_cast<long long>(M) * groups) return;
    const int m = static_cast<int>(idx / groups);
    const int q = static_cast<int>(idx % groups);
    const uint4 r = philox4x32_10(static_cast<uint32_t>(q), static_cast<uint32_t>(m), 0u, kTagInit, key);
    float* row = W + static_cast<size_t>(m) * G;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int g = q * 4 + i;
        if (g < G) row[g] = gene_from_word(word_of(r, i));
    }
}

// Device-resident state of a generation loop (game_run / game_evolve): with the seed, the first generation index, the
// running generation count and the best-fitness trace pointer in device memory, the kernels of a generation take no
// per-generation argument from the host, so the chain of one (or sixteen) generations can be captured ONCE in a CUDA graph
// and replayed (one stream, no per-generation host work).  `evals` counts the fitness finalisations of the
// run: finalisation i writes best[i] and then bumps it; the GA step that follows is step i = evals - 1.
struct RunState {
    PhiloxKey key;
    uint32_t gen0;
    int evals;
    float* best;        // [n + 1] best fitness per generation, or NULL
};

__global__ void set_run_state_kernel(RunState* run, PhiloxKey key, uint32_t gen0, float* best) {
    run->key = key;
    run->gen0 = gen0;
    run->evals = 0;
    run->best = best;
}

struct GaParams {
    int M, G, elite, tournament;
    unsigned long long t_cross, t_mut;  // Bernoulli thresholds floor(p * 2^32)
    float sigma;
    uint32_t gen;
    PhiloxKey key;
    int immigrants;                       // last R child slots are replaced by fresh random chromosomes (R12)
    int selection;                        // 0 tournament, 1 ranking, 2 roulette (R10)
    int maximize;                         // 1: fitness_dev holds 1 - error, see err_view
    const int* by_rank;                   // ranking: chromosome holding each rank (rank_kernel)
    const unsigned long long* prefix;     // roulette: inclusive prefix sums of the integer weights (roulette_prefix_kernel)
};

// ---- the paper's own selection methods ("ranking", "roulette"; defined by DESIGN.md R10).  Integer
// arithmetic only, so that the choice is bit-identical on any machine.
// floor(w * T / 2^32) for a 32-bit word and T < 2^57
__device__ __forceinline__ unsigned long long scale_word(uint32_t w, unsigned long long T) {
    return static_cast<unsigned long long>(w) * (T >> 32) + ((static_cast<unsigned long long>(w) * (T & 0xffffffffull)) >> 32);
}
// linear ranking: rank r (0 = best) has weight M - r; smallest r with C(r) = (r+1) M - r (r+1) / 2 > u
__device__ __forceinline__ int rank_from_word(uint32_t w, int M) {
    const unsigned long long Mu = static_cast<unsigned long long>(M);
    const unsigned long long u = scale_word(w, Mu * (Mu + 1) / 2);
    int lo = 0, hi = M - 1;
    while (lo < hi) {
        const unsigned long long r = static_cast<unsigned long long>((lo + hi) >> 1);
        if ((r + 1) * Mu - r * (r + 1) / 2 > u) hi = static_cast<int>(r); else lo = static_cast<int>(r) + 1;
    }
    return lo;
}
// roulette weight of a fitness: floor(clamp(1 - key(F), 0, 1) * 2^32) in double (PAPER.md:91 fitness = 1 - error)
__device__ __forceinline__ unsigned long long roulette_weight(float f) {
    const double v = 1.0 - static_cast<double>(fit_key(f));
    if (!(v > 0.0)) return 0ull;
    if (v >= 1.0) return 1ull << 32;
    return static_cast<unsigned long long>(v * 4294967296.0);
}
// smallest index whose inclusive prefix sum exceeds floor(w T / 2^32); T = 0 -> uniform index
// (`prefix` and `by_rank` are generic pointers: global memory written by an earlier kernel of the chain in ga_step_kernel,
// shared memory in ga_fused_kernel -- plain loads, which are coherent after griddepcontrol.wait.)
__device__ __forceinline__ int roulette_from_word(uint32_t w, int M, const unsigned long long* prefix) {
    const unsigned long long T = prefix[M - 1];
    if (T == 0) return static_cast<int>(index_below(w, static_cast<uint32_t>(M)));
    const unsigned long long u = scale_word(w, T);
    int lo = 0, hi = M - 1;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (prefix[mid] > u) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// by_rank[rank of chromosome c] = c; one block per chromosome (the same count as in ga_step_kernel).
__global__ void __launch_bounds__(kGaThreads) rank_kernel(const float* F, int M, int* by_rank, int maximize) {
    __shared__ int s_warp_cnt[kGaThreads / 32];
    const int c = blockIdx.x, tid = threadIdx.x;
    const float kc = fit_key(err_view(__ldcg(F + c), maximize));
    int cnt = 0;
    for (int j = tid; j < M; j += kGaThreads) cnt += precedes(fit_key(err_view(__ldcg(F + j), maximize)), j, kc, c) ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((tid & 31) == 0) s_warp_cnt[tid >> 5] = cnt;
    __syncthreads();
    if (tid == 0) {
        int r = 0;
        for (int w = 0; w < kGaThreads / 32; ++w) r += s_warp_cnt[w];
        by_rank[r] = c;
    }
}

// Inclusive prefix sums of the roulette weights; one block of 1024 threads, each owning a contiguous segment.
__global__ void __launch_bounds__(1024) roulette_prefix_kernel(const float* F, int M, unsigned long long* prefix, int maximize) {
    __shared__ unsigned long long s_tot[1024];
    const int tid = threadIdx.x;
    const int per = (M + 1023) / 1024;
    const int i0 = tid * per, i1 = min(M, i0 + per);
    unsigned long long acc = 0;
    for (int i = i0; i < i1; ++i) acc += roulette_weight(err_view(__ldcg(F + i), maximize));
    s_tot[tid] = acc;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {               // Hillis-Steele scan of the 1024 segment totals (integers: exact)
        const unsigned long long v = tid >= o ? s_tot[tid - o] : 0ull;
        __syncthreads();
        s_tot[tid] += v;
        __syncthreads();
    }
    acc = tid > 0 ? s_tot[tid - 1] : 0ull;
    for (int i = i0; i < i1; ++i) {
        acc += roulette_weight(err_view(__ldcg(F + i), maximize));
        prefix[i] = acc;
    }
}

// ---- one generation (R7).  Block c plays two parts, with no grid-wide synchronisation:
//  (1) as chromosome c of the OLD population it counts how many chromosomes precede it; if that rank is
//      below `elite` it copies its row, unchanged, to slot `rank` of the new population (elitism);
//  (2) as child slot c >= elite of the NEW population it runs the two tournaments, the crossover draw
//      and the per-gene mutation draws for that slot.
// With `img` != nullptr (tensor-core scheme, images of the OLD population valid) every gene written to the new population
// is also split into the W operand images of fitness_umma_kernel, which then needs no image pass of its own; under the
// stop rule rows carry over in place and their images stay as they are.
// W, F, stop, by_rank and prefix are written by earlier kernels of the launch chain, which may still be running when this
// grid starts (pdl.cuh): they are read with ld.global.cg after griddepcontrol.wait, never through the non-coherent path
// (no __ldg, no const __restrict__: ld.global.nc requires data that is read-only for the kernel's whole lifetime).
// The images hold every row times its own power-of-two scale (fitness_umma.cuh: the largest gene of the row lands in
// [2^13, 2^14)), so a row's images are written in a second pass, once the block knows the row's largest gene.  `amax` is
// the thread's maximum of abs_bits over the genes >= 1 it wrote; a thread's first kGaRegGenes genes (g = tid + i * 128)
// are handed over in registers, any further ones are re-read from `row` (the thread's own stores).  One barrier.
constexpr int kGaRegGenes = 4;
__device__ __forceinline__ void store_row_images(uint8_t* img, float* wscale, int img_steps, int m, const float* row, int G,
                                                 uint32_t amax, const float (&vreg)[kGaRegGenes], uint32_t* s_red) {
    const int tid = threadIdx.x;
    amax = __reduce_max_sync(0xffffffffu, amax);
    if ((tid & 31) == 0) s_red[tid >> 5] = amax;
    __syncthreads();
    amax = s_red[0];
#pragma unroll
    for (int w = 1; w < kGaThreads / 32; ++w) amax = max(amax, s_red[w]);
    const int k = umma::row_scale_exp_bits(amax);
    const float scale = ldexpf(1.0f, k);
    if (tid == 0) wscale[m] = umma::row_unscale(k);
#pragma unroll
    for (int i = 0; i < kGaRegGenes; ++i) {
        const int g = tid + i * kGaThreads;
        if (g >= 1 && g < G) umma::store_w_image_gene(img, img_steps, m, g, vreg[i] * scale);
    }
    for (int g = tid + kGaRegGenes * kGaThreads; g < G; g += kGaThreads) umma::store_w_image_gene(img, img_steps, m, g, row[g] * scale);
}

__global__ void __launch_bounds__(kGaThreads) ga_step_kernel(const float* W, const float* F, float* Wn, GaParams p,
                                                              const int* stop, uint8_t* img, float* wscale, int img_steps,
                                                              const RunState* run) {
    __shared__ int s_warp_cnt[kGaThreads / 32];
    __shared__ uint32_t s_red_elite[kGaThreads / 32], s_red_child[kGaThreads / 32];   // one per use: no barrier between them
    __shared__ int s_rank;
    __shared__ int s_parent[2];
    __shared__ int s_cut;
    const int c = blockIdx.x;
    const int tid = threadIdx.x;
    const int M = p.M, G = p.G;
    pdl_wait();                            // F (finalize), W and, for ranking / roulette, by_rank / prefix are complete
    pdl_launch_dependents();
    if (run != nullptr) {                  // generation loop replayed from a graph: seed and generation index live on the device
        p.key.k0 = __ldcg(&run->key.k0);
        p.key.k1 = __ldcg(&run->key.k1);
        p.gen = __ldcg(&run->gen0) + static_cast<uint32_t>(__ldcg(&run->evals) - 1);
    }
    if (stop != nullptr && __ldcg(stop) != 0) {   // stop rule already met: the population is final, carry it over unchanged
        for (int g = tid; g < G; g += kGaThreads) Wn[static_cast<size_t>(c) * G + g] = __ldcg(W + static_cast<size_t>(c) * G + g);
        return;
    }

    // (1) rank of chromosome c under the order
    const float kc = fit_key(err_view(__ldcg(F + c), p.maximize));
    int cnt = 0;
    for (int j = tid; j < M; j += kGaThreads) cnt += precedes(fit_key(err_view(__ldcg(F + j), p.maximize)), j, kc, c) ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((tid & 31) == 0) s_warp_cnt[tid >> 5] = cnt;
    __syncthreads();
    if (tid == 0) {
        int r = 0;
        for (int w = 0; w < kGaThreads / 32; ++w) r += s_warp_cnt[w];
        s_rank = r;
    }
    __syncthreads();
    const int rank = s_rank;
    if (rank < p.elite) {
        const float* src = W + static_cast<size_t>(c) * G;
        float* dst = Wn + static_cast<size_t>(rank) * G;
        uint32_t amax = 0u;
        float vreg[kGaRegGenes] = {0.f, 0.f, 0.f, 0.f};
        for (int g = tid, i = 0; g < G; g += kGaThreads, ++i) {
            const float v = __ldcg(src + g);
            dst[g] = v;
            if (i < kGaRegGenes) vreg[i] = v;
            if (g >= 1) amax = max(amax, umma::abs_bits(v));
        }
        if (img != nullptr) store_row_images(img, wscale, img_steps, rank, dst, G, amax, vreg, s_red_elite);
    }
    if (c < p.elite) return;  // slots 0..elite-1 are written by the elites themselves
    if (c >= M - p.immigrants) {
        // random replacement: genes uniform in [-1,1) as at initialisation, tag IMMIGRANT
        float* fresh = Wn + static_cast<size_t>(c) * G;
        uint32_t amax = 0u;
        float vreg[kGaRegGenes] = {0.f, 0.f, 0.f, 0.f};
        for (int g = tid, i = 0; g < G; g += kGaThreads, ++i) {
            const uint4 r = philox4x32_10(static_cast<uint32_t>(g >> 2), static_cast<uint32_t>(c), p.gen, kTagImmigrant, p.key);
            const float v = gene_from_word(word_of(r, g & 3));
            fresh[g] = v;
            if (i < kGaRegGenes) vreg[i] = v;
            if (g >= 1) amax = max(amax, umma::abs_bits(v));
        }
        if (img != nullptr) store_row_images(img, wscale, img_steps, c, fresh, G, amax, vreg, s_red_child);
        return;
    }

    // (2) tournaments: entrants 0..k-1 -> parent A, k..2k-1 -> parent B (with replacement).  The first warp draws the
    // entrants in parallel (one per lane: a Philox block and a fitness load each, which one thread used to do one after
    // the other) and takes the minimum of each side under the order -- a minimum, so the result is that of the sequential
    // scan; lane 31 draws the crossover meanwhile.
    if (tid < 32) {
        const int k = p.tournament;
        float bkey[2] = {INFINITY, INFINITY};
        int bidx[2] = {0x7fffffff, 0x7fffffff};
        if (p.selection == 0) {
            for (int e = tid; e < 2 * k; e += 32) {
                const uint4 r = philox4x32_10(static_cast<uint32_t>(e >> 2), static_cast<uint32_t>(c), p.gen, kTagSelect, p.key);
                const int idx = static_cast<int>(index_below(word_of(r, e & 3), static_cast<uint32_t>(M)));
                const float ki = fit_key(err_view(__ldcg(F + idx), p.maximize));
                const int side = e < k ? 0 : 1;
                if (precedes(ki, idx, bkey[side], bidx[side])) {
                    bkey[side] = ki;
                    bidx[side] = idx;
                }
            }
#pragma unroll
            for (int side = 0; side < 2; ++side)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const float ok = __shfl_xor_sync(0xffffffffu, bkey[side], o);
                    const int oi = __shfl_xor_sync(0xffffffffu, bidx[side], o);
                    if (precedes(ok, oi, bkey[side], bidx[side])) {
                        bkey[side] = ok;
                        bidx[side] = oi;
                    }
                }
        } else if (tid == 0) {
            // ranking / roulette: parents A and B from words 0 and 1 of one SELECT draw
            const uint4 r = philox4x32_10(0u, static_cast<uint32_t>(c), p.gen, kTagSelect, p.key);
            if (p.selection == 1) {
                bidx[0] = p.by_rank[rank_from_word(r.x, M)];
                bidx[1] = p.by_rank[rank_from_word(r.y, M)];
            } else {
                bidx[0] = roulette_from_word(r.x, M, p.prefix);
                bidx[1] = roulette_from_word(r.y, M, p.prefix);
            }
        }
        if (tid == 0) {
            s_parent[0] = bidx[0];
            s_parent[1] = bidx[1];
        }
        if (tid == 31) {
            // single-point crossover: child = A[0:q] ++ B[q:G], q in [1, G-1]; otherwise child = A
            const uint4 rc = philox4x32_10(0u, static_cast<uint32_t>(c), p.gen, kTagCross, p.key);
            int q = G;
            if (static_cast<unsigned long long>(rc.x) < p.t_cross && G >= 2)
                q = 1 + static_cast<int>(index_below(rc.y, static_cast<uint32_t>(G - 1)));
            s_cut = q;
        }
    }
    __syncthreads();
    const float* A = W + static_cast<size_t>(s_parent[0]) * G;
    const float* B = W + static_cast<size_t>(s_parent[1]) * G;
    const int q = s_cut;
    float* child = Wn + static_cast<size_t>(c) * G;
    // per-gene Gaussian mutation, no clamping (D6)
    uint32_t amax = 0u;
    float vreg[kGaRegGenes] = {0.f, 0.f, 0.f, 0.f};
    auto gene = [&](int g) {
        float v = __ldcg(g < q ? A + g : B + g);
        const uint4 rm = philox4x32_10(static_cast<uint32_t>(g), static_cast<uint32_t>(c), p.gen, kTagMutate, p.key);
        if (static_cast<unsigned long long>(rm.x) < p.t_mut) {
            const float z = gauss_from_words(rm.y, rm.z);
            v = __fadd_rn(v, __fmul_rn(p.sigma, z));
        }
        child[g] = v;
        if (g >= 1) amax = max(amax, umma::abs_bits(v));
        return v;
    };
#pragma unroll
    for (int i = 0; i < kGaRegGenes; ++i) {
        const int g = tid + i * kGaThreads;
        if (g < G) vreg[i] = gene(g);
    }
    for (int g = tid + kGaRegGenes * kGaThreads; g < G; g += kGaThreads) gene(g);
    if (img != nullptr) store_row_images(img, wscale, img_steps, c, child, G, amax, vreg, s_red_child);
}

// ---- fitness finalisation: F[m] = (sum over partial rows, in row order) / P in fp64, rounded to fp32
// (PAPER.md:63 MSE).  Optionally the best (lowest, NaN worst, ties -> lower index) fitness of the
// population is written to *best_out by the last block to finish (R8).
constexpr int kFinThreads = 1024, kFinCols = 32, kFinGroups = kFinThreads / kFinCols;

__global__ void __launch_bounds__(kFinThreads) finalize_fitness_kernel(const double* part, int n_part, int m_stride, int M,
                                                                        double P_d, float* F, double* sse_out, float* best_out,
                                                                        float* blk_key, int* blk_idx, unsigned int* ticket,
                                                                        int* stop, float threshold, int gen_index, int metric,
                                                                        RunState* run, int part_ff) {
    __shared__ float s_key[kFinThreads / 32];
    __shared__ int s_idx[kFinThreads / 32];
    __shared__ bool s_last;
    // 32 chromosomes per block x 32 row groups: row group g sums partial rows g, g+32, g+64, ... with four independent
    // accumulators (the loads are L2 latency-bound: one thread walking all ~300 rows took 108 us at M = 4096; 8 groups
    // 15 us, of which ten dependent L2 round trips), then the 32 group sums are added in group order -- a fixed order, so the
    // result is bit-stable.
    pdl_wait();                                    // the fitness kernel's partial sums are complete
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;   // stop rule met earlier: fitness and best trace stay as they are
    __shared__ double s_grp[kFinGroups][kFinCols];
    const int col = threadIdx.x % kFinCols, grp = threadIdx.x / kFinCols;
    const int m = blockIdx.x * kFinCols + col;
    float key = INFINITY;
    int idx = 0x7fffffff;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    if (m < M && !part_ff) {          // FFMA kernel: a partial row holds fp64 sums
        int r = grp;
        for (; r + 3 * kFinGroups < n_part; r += 4 * kFinGroups) {
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[i] += __ldcg(part + static_cast<size_t>(r + i * kFinGroups) * m_stride + m);
        }
#pragma unroll
        for (int i = 0; i < 3; ++i)      // the tail: at most three rows, same accumulator per position as above
            if (r + i * kFinGroups < n_part) acc[i] += __ldcg(part + static_cast<size_t>(r + i * kFinGroups) * m_stride + m);
    } else if (m < M) {
        // tensor-core kernel: float-float pairs (hi, lo) in the same 8 bytes.  They are added in float-float arithmetic
        // too (error-free TwoSum of the hi parts, the lo parts and the errors in a second fp32 sum) and widened to fp64
        // once per accumulator: an fp64 add per row made this kernel 4 us slower (fp64 is a slow pipe on this chip).
        float ah[4] = {0.f, 0.f, 0.f, 0.f}, al[4] = {0.f, 0.f, 0.f, 0.f};
        auto add = [&](int i, int row) {
            const float2 v = __ldcg(reinterpret_cast<const float2*>(part + static_cast<size_t>(row) * m_stride + m));
            const float hi = __fadd_rn(ah[i], v.x);
            const float bv = __fadd_rn(hi, -ah[i]);
            const float er = __fadd_rn(__fadd_rn(ah[i], -__fadd_rn(hi, -bv)), __fadd_rn(v.x, -bv));
            ah[i] = hi;
            al[i] = __fadd_rn(al[i], __fadd_rn(v.y, er));
        };
        int r = grp;
        for (; r + 3 * kFinGroups < n_part; r += 4 * kFinGroups) {
#pragma unroll
            for (int i = 0; i < 4; ++i) add(i, r + i * kFinGroups);
        }
#pragma unroll
        for (int i = 0; i < 3; ++i)
            if (r + i * kFinGroups < n_part) add(i, r + i * kFinGroups);
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[i] = static_cast<double>(ah[i]) + static_cast<double>(al[i]);
    }
    s_grp[grp][col] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
    __syncthreads();
    if (m < M && grp == 0) {
        double s = 0.0;
#pragma unroll
        for (int g = 0; g < kFinGroups; ++g) s += s_grp[g][col];
        if (sse_out != nullptr) {            // pattern-sharded evaluation: hand out the un-normalised sum instead
            sse_out[m] = s;
        } else {
            // MSE or RMSE; or the fitness 1 - error (metric 2), whose order is taken on the error
            const float f = static_cast<float>(metric == 1 ? sqrt(s / P_d) : (metric == 2 ? 1.0 - s / P_d : s / P_d));
            F[m] = f;
            key = fit_key(err_view(f, metric == 2));
            idx = m;
        }
    }
    if (sse_out != nullptr) return;
    if (best_out == nullptr && run == nullptr) return;
    __threadfence();  // F[m] visible device-wide before this block takes its ticket
    auto warp_min = [](float& k, int& i) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ok = __shfl_xor_sync(0xffffffffu, k, o);
            const int oi = __shfl_xor_sync(0xffffffffu, i, o);
            if (precedes(ok, oi, k, i)) {
                k = ok;
                i = oi;
            }
        }
    };
    warp_min(key, idx);
    if ((threadIdx.x & 31) == 0) {
        s_key[threadIdx.x >> 5] = key;
        s_idx[threadIdx.x >> 5] = idx;
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        key = threadIdx.x < kFinThreads / 32 ? s_key[threadIdx.x] : INFINITY;
        idx = threadIdx.x < kFinThreads / 32 ? s_idx[threadIdx.x] : 0x7fffffff;
        warp_min(key, idx);
        if (threadIdx.x == 0) {
            blk_key[blockIdx.x] = key;
            blk_idx[blockIdx.x] = idx;
            __threadfence();
            const unsigned int t = atomicAdd(ticket, 1u);
            s_last = (t == gridDim.x - 1);
        }
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x < 32) {
        key = INFINITY;
        idx = 0x7fffffff;
        for (int b = threadIdx.x; b < static_cast<int>(gridDim.x); b += 32) {
            const float ok = __ldcg(blk_key + b);
            const int oi = __ldcg(blk_idx + b);
            if (precedes(ok, oi, key, idx)) {
                key = ok;
                idx = oi;
            }
        }
        warp_min(key, idx);
        if (threadIdx.x == 0) {
            const float best = __ldcg(F + idx);  // the fitness itself (NaN if every chromosome is NaN: idx = 0)
            if (run != nullptr) {                // graph replay: the trace slot comes from the device-side generation count
                const int evals = __ldcg(&run->evals);
                float* base = reinterpret_cast<float*>(__ldcg(reinterpret_cast<unsigned long long*>(&run->best)));
                best_out = base != nullptr ? base + evals : nullptr;
                run->evals = evals + 1;          // nobody reads it until the next kernel of the chain
            }
            if (best_out != nullptr) *best_out = best;
            *ticket = 0u;
            if (stop != nullptr) {
                stop[1] = gen_index;                       // GA steps performed so far
                if (err_view(best, metric == 2) <= threshold) stop[0] = 1;   // learning-error threshold reached
            }
        }
    }
}

}  // namespace game
