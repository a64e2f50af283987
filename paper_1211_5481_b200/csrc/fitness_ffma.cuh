// Fused fitness on the CUDA cores (scheme GAME_SCHEME_FFMA): the minimum-slice kernel and the path for
// shapes the tensor-core kernel does not cover.  One block = one tile of 128 patterns:
//   expansion phi(x) into shared memory (eq.(1) Chebyshev by recurrence
//   eq.(6) trig by one accurate sincos per feature + multiple-angle recurrences), never written to HBM;
//   z = W . phi (eq.(2)) in fp32 FFMA, 8 chromosomes per pass; activation (D2);
//   squared error (eq.(3)); per-chromosome sum over the tile (warp shuffles, fixed order)
//   accumulated in fp64 into this block's private row of `part` (no atomics => bit-stable).
#pragma once
#include <cstdint>

#include "pdl.cuh"

namespace game {

constexpr int kFfmaTile = 128;   // patterns per tile == threads per block
constexpr int kFfmaMB = 8;       // chromosomes per pass
constexpr int kFfmaMaxG = 448;   // phi tile = G * 128 floats <= 224 KB

__device__ __forceinline__ float activate(int act, float z) {
    if (act == 1) {  // sigmoid = 1 / (1 + 2^(-z log2 e)); saturates to 0 / 1, NaN only for NaN z
        return __frcp_rn(1.0f + exp2f(-1.44269504088896340736f * z));
    }
    if (act == 2) {  // tanh = 1 - 2 / (1 + 2^(2 z log2 e))
        return 1.0f - 2.0f * __frcp_rn(1.0f + exp2f(2.88539008177792681472f * z));
    }
    return z;
}

// phi(x) of ONE pattern into dst[g * stride] (gene order of include/game.h).  shared = the paper's literal form
// (eq.(2), 75-77 eq.(5)): one coefficient per degree for ALL features, so the term of gene j is the sum
// over the features of g_j(f_i) -- the per-pattern sums of cosines / sines the paper precomputes.
__device__ __forceinline__ void expand_pattern(const float* __restrict__ xr, bool valid, int N, int d, int expansion,
                                               int shared, float* __restrict__ dst, int stride) {
    dst[0] = 1.0f;  // gene 0: bias a_0
    const int terms = expansion == 0 ? d : 2 * d;
    if (shared)
        for (int g = 1; g <= terms; ++g) dst[g * stride] = 0.0f;
    for (int i = 0; i < N; ++i) {
        const float x = valid ? xr[i] : 0.0f;
        float* blk = dst + (1 + (shared ? 0 : i * terms)) * stride;
        if (expansion == 0) {
            const float x2 = 2.0f * x;
            float tm = 1.0f, tc = x;
            for (int j = 0; j < d; ++j) {
                blk[j * stride] = shared ? blk[j * stride] + tc : tc;
                const float tn = fmaf(x2, tc, -tm);
                tm = tc;
                tc = tn;
            }
        } else {
            float s1, c1;
            sincosf(x, &s1, &c1);
            const float x2 = 2.0f * c1;
            float cm = 1.0f, cc = c1, sm = 0.0f, sc = s1;
            for (int k = 0; k < d; ++k) {
                blk[k * stride] = shared ? blk[k * stride] + cc : cc;
                blk[(d + k) * stride] = shared ? blk[(d + k) * stride] + sc : sc;
                const float cn = fmaf(x2, cc, -cm), sn = fmaf(x2, sc, -sm);
                cm = cc; cc = cn;
                sm = sc; sc = sn;
            }
        }
    }
}

// X and t are never written by the library's kernels (non-coherent loads are fine); W and the stop flag are written by
// earlier kernels of the launch chain (pdl.cuh) and are read with ld.global.cg after griddepcontrol.wait.
__global__ void __launch_bounds__(kFfmaTile) fitness_ffma_kernel(const float* __restrict__ X,
                                                                  const float* __restrict__ t,
                                                                  const float* W, double* part, long long P, int N,
                                                                  int d, int M, int G, int expansion, int act,
                                                                  int m_stride, long long n_tiles, const int* stop, int shared) {
    pdl_wait();                // W, the partial sums and the stop flag are complete (pdl.cuh)
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;
    extern __shared__ float phi[];  // [G][128]
    __shared__ float s_wsum[kFfmaTile / 32][kFfmaMB];
    const int tid = threadIdx.x;
    double* my_part = part + static_cast<size_t>(blockIdx.x) * m_stride;
    for (int m = tid; m < m_stride; m += kFfmaTile) my_part[m] = 0.0;
    __syncthreads();

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long p = tile * kFfmaTile + tid;
        const bool valid = p < P;
        const float* xr = X + (valid ? p : 0) * N;
        expand_pattern(xr, valid, N, d, expansion, shared, phi + tid, kFfmaTile);
        const float tp = valid ? t[p] : 0.0f;
        __syncthreads();

        for (int m0 = 0; m0 < M; m0 += kFfmaMB) {
            float z[kFfmaMB];
            const float* wrow[kFfmaMB];
#pragma unroll
            for (int i = 0; i < kFfmaMB; ++i) {
                z[i] = 0.0f;
                const int m = m0 + i < M ? m0 + i : M - 1;
                wrow[i] = W + static_cast<size_t>(m) * G;
            }
            for (int g = 0; g < G; ++g) {
                const float ph = phi[g * kFfmaTile + tid];
#pragma unroll
                for (int i = 0; i < kFfmaMB; ++i) z[i] = fmaf(__ldcg(wrow[i] + g), ph, z[i]);
            }
#pragma unroll
            for (int i = 0; i < kFfmaMB; ++i) {
                const float e = valid ? activate(act, z[i]) - tp : 0.0f;
                float e2 = e * e;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
                if ((tid & 31) == 0) s_wsum[tid >> 5][i] = e2;
            }
            __syncthreads();
            if (tid < kFfmaMB && m0 + tid < M) {
                const float s = (s_wsum[0][tid] + s_wsum[1][tid]) + (s_wsum[2][tid] + s_wsum[3][tid]);
                my_part[m0 + tid] += static_cast<double>(s);
            }
            __syncthreads();
        }
    }
}

}  // namespace game
