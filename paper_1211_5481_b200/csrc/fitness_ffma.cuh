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
// earlier kernels of the launch chain (pdl.cuh) and are read with plain / ld.global.cg loads after griddepcontrol.wait.
//
// Register tile: a thread owns 4 consecutive patterns x 8 chromosomes (32 accumulators); a warp covers the tile's 128
// patterns for ITS 8 chromosomes, the block's eight warps take eight chromosome groups, i.e. 64 chromosomes per pass.  Per
// gene a thread issues one 16-byte shared load of phi, two warp-uniform 16-byte loads of the TRANSPOSED W (L1 / L2 hits)
// and 32 FFMAs -- the first version (1 pattern x 8 chromosomes per thread) issued 8 scalar loads for 8 FFMAs and was bound
// by the load pipe at 13 % of the FFMA peak.  A chromosome's sum over the tile is a fixed-order shuffle reduction inside the
// one warp that owns it: no shared-memory staging, no block barrier per pass.
// W [M][G] -> Wt [G][m_stride] (rows past M zero): the 8 chromosomes of a warp at one gene are then 32 contiguous bytes
// (two 16-byte loads instead of eight scalar ones).  Runs before every FFMA evaluation; 32 x 32 tiles through shared memory.
__global__ void __launch_bounds__(256) ffma_transpose_kernel(const float* W, float* Wt, int M, int G, int m_stride) {
    __shared__ float tile[32][33];
    pdl_wait();                // W is complete, and so is the evaluation that read the old transpose
    pdl_launch_dependents();
    const int g0 = blockIdx.x * 32, m0 = blockIdx.y * 32, tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, g = g0 + tx;
        tile[r][tx] = (m < M && g < G) ? __ldcg(W + static_cast<size_t>(m) * G + g) : 0.0f;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int g = g0 + r, m = m0 + tx;
        if (g < G && m < m_stride) Wt[static_cast<size_t>(g) * m_stride + m] = tile[tx][r];
    }
}

constexpr int kFfmaPT = 4;                       // patterns per thread
constexpr int kFfmaThreads = 256;                // 8 warps: the first four also expand the tile's patterns
constexpr int kFfmaWarps = kFfmaThreads / 32;    // chromosome groups per pass
static_assert(kFfmaTile == 32 * kFfmaPT, "a warp covers the tile's patterns, kFfmaPT per lane");
static_assert(kFfmaMB == 8, "two float4 of the transposed W per gene");

__global__ void __launch_bounds__(kFfmaThreads) fitness_ffma_kernel(const float* __restrict__ X,
                                                                  const float* __restrict__ t,
                                                                  const float* Wt, double* part, long long P, int N,
                                                                  int d, int M, int G, int expansion, int act,
                                                                  int m_stride, long long n_tiles, const int* stop, int shared) {
    pdl_wait();                // the transposed W, the partial sums and the stop flag are complete (pdl.cuh)
    pdl_launch_dependents();
    if (stop != nullptr && __ldcg(stop) != 0) return;
    extern __shared__ __align__(16) float phi[];  // [G][128]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double* my_part = part + static_cast<size_t>(blockIdx.x) * m_stride;
    for (int m = tid; m < m_stride; m += kFfmaThreads) my_part[m] = 0.0;
    __syncthreads();

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        if (tid < kFfmaTile) {   // expansion: one thread per pattern of the tile
            const long long p = tile * kFfmaTile + tid;
            const bool valid = p < P;
            expand_pattern(X + (valid ? p : 0) * N, valid, N, d, expansion, shared, phi + tid, kFfmaTile);
        }
        // this thread's 4 patterns (columns 4 lane .. 4 lane + 3 of the tile) and their targets
        const long long p0 = tile * kFfmaTile + kFfmaPT * lane;
        float tp[kFfmaPT];
        bool valid[kFfmaPT];
#pragma unroll
        for (int j = 0; j < kFfmaPT; ++j) {
            valid[j] = p0 + j < P;
            tp[j] = valid[j] ? __ldg(t + p0 + j) : 0.0f;
        }
        __syncthreads();

        for (int m0 = warp * kFfmaMB; m0 < M; m0 += kFfmaWarps * kFfmaMB) {
            float z[kFfmaMB][kFfmaPT];
#pragma unroll
            for (int i = 0; i < kFfmaMB; ++i)
#pragma unroll
                for (int j = 0; j < kFfmaPT; ++j) z[i][j] = 0.0f;
            const float4* wcol = reinterpret_cast<const float4*>(Wt + m0);      // + g * m_stride: this warp's 8 chromosomes at gene g
            const int wstep = m_stride / 4;
#pragma unroll 4
            for (int g = 0; g < G; ++g) {
                const float4 ph = *reinterpret_cast<const float4*>(phi + g * kFfmaTile + kFfmaPT * lane);
                const float4 wa = wcol[static_cast<size_t>(g) * wstep], wb = wcol[static_cast<size_t>(g) * wstep + 1];   // warp-uniform, coherent (plain loads after the wait)
                const float wv[kFfmaMB] = {wa.x, wa.y, wa.z, wa.w, wb.x, wb.y, wb.z, wb.w};
#pragma unroll
                for (int i = 0; i < kFfmaMB; ++i) {
                    const float w = wv[i];
                    z[i][0] = fmaf(w, ph.x, z[i][0]);
                    z[i][1] = fmaf(w, ph.y, z[i][1]);
                    z[i][2] = fmaf(w, ph.z, z[i][2]);
                    z[i][3] = fmaf(w, ph.w, z[i][3]);
                }
            }
#pragma unroll
            for (int i = 0; i < kFfmaMB; ++i) {
                float e2 = 0.0f;
#pragma unroll
                for (int j = 0; j < kFfmaPT; ++j) {
                    const float e = valid[j] ? activate(act, z[i][j]) - tp[j] : 0.0f;
                    e2 = fmaf(e, e, e2);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) e2 += __shfl_xor_sync(0xffffffffu, e2, o);
                if (lane == 0 && m0 + i < M) my_part[m0 + i] += static_cast<double>(e2);   // this warp owns chromosome m0 + i
            }
        }
        __syncthreads();            // the next tile's expansion overwrites phi
    }
}

}  // namespace game
