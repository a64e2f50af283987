// The whole generation loop in ONE persistent kernel, for the latency-bound regime the paper's own experiments live
// in (2100 patterns, a few dozen chromosomes, thousands of iterations; "time linear in
// iterations").  At that size a generation is ~6 MFLOP: five kernel launches per generation (38 us)
// are all overhead.  Here the grid (one CTA per SM, launched cooperatively so that all CTAs are co-resident) keeps
// going for n generations with two grid barriers per generation:
//
//   setup      : each CTA expands ITS slice of the patterns once (phi in shared memory; X never changes)
//   per generation
//     phase 1  : partial sums of squared errors of every chromosome over the CTA's patterns (fp32 FFMA, one warp per
//                chromosome, fixed shuffle tree)                                      -> part[cta][m]   | grid barrier
//     phase 2  : every CTA adds the partial rows in row order (identical result everywhere), ranks the chromosomes,
//                and builds the child slots c = cta, cta + grid, ... exactly as ga_step_kernel does (same Philox
//                counters, same integer maps, same exact-op Gaussian)                  -> the other buffer | grid barrier
//
// Arithmetic = the FFMA scheme's (fp32 recurrences and dot products): fitness within 1e-5 of the oracle, operators
// bit-exact given the fitness vector the kernel itself produced.
#pragma once
#include <cstdint>

#include "fitness_ffma.cuh"
#include "ga_kernels.cuh"

namespace game {

constexpr int kFusedThreads = 256;
constexpr int kFusedMaxM = 1024;

struct FusedParams {
    const float* X;
    const float* t;
    float* pop[2];            // population buffers; pop[cur] is current at entry
    float* F;                 // [M] fitness of the LAST evaluated generation
    double* part;             // [gridDim.x][M]
    float* best;              // [n_gens] best fitness of every evaluated generation, or NULL
    unsigned int* barrier;    // zeroed by the host before the launch
    long long P;
    int N, d, M, G, expansion, act, rmse, shared;
    int cur, n_gens, ppc;     // ppc = patterns per CTA (contiguous slices)
    GaParams ga;              // gen = first generation index
};

// All CTAs arrive; thread 0 of each spins until everyone of this epoch has.  The counter only grows within a launch
// (the host zeroes it and caps a launch at 2^20 generations, so it cannot wrap); the wait is bounded in TIME (20 s of
// globaltimer: a protocol bug traps instead of hanging the GPU, time-slicing or a debugger cannot trip it).
__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int& epoch) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        epoch += gridDim.x;
        atomicAdd(counter, 1u);
        unsigned int n = 0;
        unsigned long long t0 = 0;
        while (*reinterpret_cast<volatile unsigned int*>(counter) < epoch) {
            if ((++n & 0xffffu) == 0) {
                const unsigned long long now = global_timer_ns();
                if (t0 == 0) t0 = now;
                else if (now - t0 > 20000000000ull) __trap();
            }
        }
        __threadfence();
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kFusedThreads, 1) ga_fused_kernel(const FusedParams prm) {
    extern __shared__ __align__(16) unsigned char fused_smem[];
    const int M = prm.M, G = prm.G, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // shared memory: phi[ppc][G], Ws[M][G], tl[ppc], Fs[M], by_rank[M], prefix[M]
    float* phi = reinterpret_cast<float*>(fused_smem);
    float* Ws = phi + static_cast<size_t>(prm.ppc) * G;
    float* tl = Ws + static_cast<size_t>(M) * G;
    float* Fs = tl + prm.ppc;
    int* by_rank = reinterpret_cast<int*>(Fs + M);
    unsigned long long* prefix = reinterpret_cast<unsigned long long*>(
        (reinterpret_cast<uintptr_t>(by_rank + M) + 7) & ~static_cast<uintptr_t>(7));
    __shared__ int s_parent[2];
    __shared__ int s_cut;
    __shared__ double s_grp[kFusedThreads / 32][32];

    const long long p_begin = static_cast<long long>(blockIdx.x) * prm.ppc;
    const int n_mine = static_cast<int>(max(0ll, min(static_cast<long long>(prm.ppc), prm.P - p_begin)));

    // ---- setup: expansion of this CTA's patterns, once (gene order of include/game.h)
    for (int q = tid; q < n_mine; q += kFusedThreads) {
        const float* xr = prm.X + (p_begin + q) * prm.N;
        expand_pattern(xr, true, prm.N, prm.d, prm.expansion, prm.shared, phi + static_cast<size_t>(q) * G, 1);
        tl[q] = __ldg(prm.t + p_begin + q);
    }
    __syncthreads();

    unsigned int epoch = 0;
    int cur = prm.cur;
    double* my_part = prm.part + static_cast<size_t>(blockIdx.x) * M;
    GaParams ga = prm.ga;
    ga.by_rank = by_rank;
    ga.prefix = prefix;

    for (int it = 0; it < prm.n_gens; ++it, ++ga.gen) {
        const float* W = prm.pop[cur];
        float* Wn = prm.pop[cur ^ 1];
        // the population of this generation, staged in shared memory (written by other CTAs: bypass L1)
        for (int i = tid; i < M * G; i += kFusedThreads) Ws[i] = __ldcg(W + i);
        __syncthreads();
        // ---- phase 1: one warp per chromosome, lanes over this CTA's patterns
        for (int m = warp; m < M; m += kFusedThreads / 32) {
            const float* w = Ws + static_cast<size_t>(m) * G;
            float acc = 0.0f;
            for (int q = lane; q < n_mine; q += 32) {
                const float* row = phi + static_cast<size_t>(q) * G;
                float z = 0.0f;
                for (int g = 0; g < G; ++g) z = fmaf(w[g], row[g], z);
                const float e = activate(prm.act, z) - tl[q];
                acc = fmaf(e, e, acc);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) __stcg(my_part + m, static_cast<double>(acc));
        }
        grid_barrier(prm.barrier, epoch);

        // ---- phase 2a: fitness (identical in every CTA: same rows, same order).  32 chromosomes at a time, 8 row groups
        // with 4 independent accumulators each (the loads are L2-latency bound), groups added in group order.
        for (int m0 = 0; m0 < M; m0 += 32) {
            const int col = tid & 31, grp = tid >> 5, m = m0 + col;
            double acc[4] = {0.0, 0.0, 0.0, 0.0};
            if (m < M) {
                unsigned int r = grp;
                for (; r + 24 < gridDim.x; r += 32) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) acc[i] += __ldcg(prm.part + static_cast<size_t>(r + 8 * i) * M + m);
                }
                for (int i = 0; r < gridDim.x; r += 8, ++i) acc[i] += __ldcg(prm.part + static_cast<size_t>(r) * M + m);
            }
            s_grp[grp][col] = (acc[0] + acc[1]) + (acc[2] + acc[3]);
            __syncthreads();
            if (grp == 0 && m < M) {
                double s = 0.0;
#pragma unroll
                for (int g = 0; g < 8; ++g) s += s_grp[g][col];
                const double mse = s / static_cast<double>(prm.P);
                Fs[m] = static_cast<float>(prm.rmse == 1 ? sqrt(mse) : (prm.rmse == 2 ? 1.0 - mse : mse));
            }
            __syncthreads();
        }
        // ranks (chromosome per rank) and roulette prefix sums, in shared memory
        for (int m = tid; m < M; m += kFusedThreads) {
            const float km = fit_key(err_view(Fs[m], ga.maximize));
            int r = 0;
            for (int j = 0; j < M; ++j) r += precedes(fit_key(err_view(Fs[j], ga.maximize)), j, km, m) ? 1 : 0;
            by_rank[r] = m;
        }
        if (ga.selection == 2 && tid == 0) {
            unsigned long long a = 0;
            for (int m = 0; m < M; ++m) {
                a += roulette_weight(err_view(Fs[m], ga.maximize));
                prefix[m] = a;
            }
        }
        __syncthreads();
        if (blockIdx.x == 0) {
            for (int m = tid; m < M; m += kFusedThreads) prm.F[m] = Fs[m];
            if (tid == 0 && prm.best != nullptr) prm.best[it] = Fs[by_rank[0]];
        }
        // ---- phase 2b: child slots of this CTA (the logic of ga_step_kernel, fitness and ranks from shared memory)
        for (int c = blockIdx.x; c < M; c += gridDim.x) {
            float* child = Wn + static_cast<size_t>(c) * G;
            if (c < ga.elite) {                                    // elitism: rank c, bit-copied
                const float* src = Ws + static_cast<size_t>(by_rank[c]) * G;
                for (int g = tid; g < G; g += kFusedThreads) child[g] = src[g];
                continue;
            }
            if (c >= M - ga.immigrants) {                          // random replacement (R12)
                for (int g = tid; g < G; g += kFusedThreads) {
                    const uint4 r = philox4x32_10(static_cast<uint32_t>(g >> 2), static_cast<uint32_t>(c), ga.gen, kTagImmigrant, ga.key);
                    child[g] = gene_from_word(word_of(r, g & 3));
                }
                continue;
            }
            __syncthreads();                                       // s_parent / s_cut of the previous slot are consumed
            if (tid == 0) {
                int par[2] = {-1, -1};
                if (ga.selection == 0) {
                    float pkey[2] = {0.f, 0.f};
                    uint4 r = make_uint4(0, 0, 0, 0);
                    for (int e = 0; e < 2 * ga.tournament; ++e) {
                        if ((e & 3) == 0)
                            r = philox4x32_10(static_cast<uint32_t>(e >> 2), static_cast<uint32_t>(c), ga.gen, kTagSelect, ga.key);
                        const int idx = static_cast<int>(index_below(word_of(r, e & 3), static_cast<uint32_t>(M)));
                        const float ki = fit_key(err_view(Fs[idx], ga.maximize));
                        const int side = e < ga.tournament ? 0 : 1;
                        if (par[side] < 0 || precedes(ki, idx, pkey[side], par[side])) {
                            par[side] = idx;
                            pkey[side] = ki;
                        }
                    }
                } else {
                    const uint4 r = philox4x32_10(0u, static_cast<uint32_t>(c), ga.gen, kTagSelect, ga.key);
                    if (ga.selection == 1) {
                        par[0] = by_rank[rank_from_word(r.x, M)];
                        par[1] = by_rank[rank_from_word(r.y, M)];
                    } else {
                        par[0] = roulette_from_word(r.x, M, prefix);
                        par[1] = roulette_from_word(r.y, M, prefix);
                    }
                }
                s_parent[0] = par[0];
                s_parent[1] = par[1];
                const uint4 rc = philox4x32_10(0u, static_cast<uint32_t>(c), ga.gen, kTagCross, ga.key);
                int q = G;
                if (static_cast<unsigned long long>(rc.x) < ga.t_cross && G >= 2)
                    q = 1 + static_cast<int>(index_below(rc.y, static_cast<uint32_t>(G - 1)));
                s_cut = q;
            }
            __syncthreads();
            const float* A = Ws + static_cast<size_t>(s_parent[0]) * G;
            const float* B = Ws + static_cast<size_t>(s_parent[1]) * G;
            const int q = s_cut;
            for (int g = tid; g < G; g += kFusedThreads) {
                float v = g < q ? A[g] : B[g];
                const uint4 rm = philox4x32_10(static_cast<uint32_t>(g), static_cast<uint32_t>(c), ga.gen, kTagMutate, ga.key);
                if (static_cast<unsigned long long>(rm.x) < ga.t_mut) {
                    const float z = gauss_from_words(rm.y, rm.z);
                    v = __fadd_rn(v, __fmul_rn(ga.sigma, z));
                }
                child[g] = v;
            }
        }
        grid_barrier(prm.barrier, epoch);
        cur ^= 1;
    }
}

}  // namespace game
