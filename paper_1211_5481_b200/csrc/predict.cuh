// Test / validation use case (the trained chromosome applied to patterns; "crispy"
// classification): y[q] = act(sum_g w[g] phi_g(x_q)) for ONE chromosome over Q patterns, and the confusion counts
// of the thresholded outputs.  M = 1, so this is not a tensor-core problem: one thread per pattern, the expansion
// by recurrence fused with the dot product, fp32 FFMA; bound: HBM (4 (N + 1) bytes per pattern).
#pragma once
#include <cstdint>

#include "fitness_ffma.cuh"

namespace game {

constexpr int kPredictThreads = 256;

__global__ void __launch_bounds__(kPredictThreads) predict_kernel(const float* __restrict__ X, const float* __restrict__ w,
                                                                   float* __restrict__ y, long long Q, int N, int d, int G,
                                                                   int expansion, int act, int shared, int stage_w) {
    extern __shared__ float s_stage[];   // [G] when stage_w: the chromosome staged in shared memory (G up to 57 K genes);
                                         // longer chromosomes are read through L1 / L2 (every thread walks the same genes)
    const float* s_w = w;
    if (stage_w) {
        for (int g = threadIdx.x; g < G; g += kPredictThreads) s_stage[g] = w[g];
        __syncthreads();
        s_w = s_stage;
    }
    for (long long q = static_cast<long long>(blockIdx.x) * kPredictThreads + threadIdx.x; q < Q;
         q += static_cast<long long>(gridDim.x) * kPredictThreads) {
        const float* xr = X + q * N;
        float z = s_w[0];   // bias a_0
        if (expansion == 0) {
            for (int i = 0; i < N; ++i) {
                const float x = __ldg(xr + i), x2 = 2.0f * x;
                const float* wi = s_w + 1 + (shared ? 0 : i * d);           // shared: the same d coefficients for every feature
                float tm = 1.0f, tc = x;
                for (int j = 0; j < d; ++j) {
                    z = fmaf(wi[j], tc, z);
                    const float tn = fmaf(x2, tc, -tm);
                    tm = tc;
                    tc = tn;
                }
            }
        } else {
            for (int i = 0; i < N; ++i) {
                float s1, c1;
                sincosf(__ldg(xr + i), &s1, &c1);
                const float x2 = 2.0f * c1;
                const float* wi = s_w + 1 + (shared ? 0 : i * 2 * d);
                float cm = 1.0f, cc = c1, sm = 0.0f, sc = s1;
                for (int k = 0; k < d; ++k) {
                    z = fmaf(wi[k], cc, z);
                    z = fmaf(wi[d + k], sc, z);
                    const float cn = fmaf(x2, cc, -cm), sn = fmaf(x2, sc, -sm);
                    cm = cc; cc = cn;
                    sm = sc; sc = sn;
                }
            }
        }
        y[q] = activate(act, z);
    }
}

// counts = {TP, FP, TN, FN}; predicted class = (y > threshold) (NaN is not above it), true class = (t > 0.5).
__global__ void __launch_bounds__(kPredictThreads) confusion_kernel(const float* __restrict__ y, const float* __restrict__ t,
                                                                     long long Q, float threshold,
                                                                     unsigned long long* __restrict__ counts) {
    unsigned long long c[4] = {0, 0, 0, 0};
    for (long long q = static_cast<long long>(blockIdx.x) * kPredictThreads + threadIdx.x; q < Q;
         q += static_cast<long long>(gridDim.x) * kPredictThreads) {
        const bool pred = y[q] > threshold, truth = t[q] > 0.5f;
        c[pred ? (truth ? 0 : 1) : (truth ? 3 : 2)] += 1;
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        unsigned long long v = c[k];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v != 0) atomicAdd(counts + k, v);
    }
}

}  // namespace game
