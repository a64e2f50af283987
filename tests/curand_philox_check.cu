// TEST INFRASTRUCTURE (tests/test_gpu_curand.py), not product code: Philox4x32-10 blocks from NVIDIA's cuRAND device
// API, the independent library implementation SURVEY.md section 8(c) "P-RNG" names as the cross-check of the oracle's
// own Philox (the Random123 known-answer file is not in the container).  Shares nothing with oracle/ or csrc/.
//   out[i][0..3] : curand_Philox4x32_10(ctr, key), the library's block function
//   out[i][4..7] : curand_init(seed = key, subsequence = ctr2 | ctr3 << 32, offset = 4 (ctr0 | ctr1 << 32)) followed by
//                  curand4() on a curandStatePhilox4_32_10_t -- the public generator; zeros when 4 * counter overflows
#include <cuda_runtime.h>
#include <curand_kernel.h>

__global__ void philox_blocks_kernel(int n, const unsigned* __restrict__ in, unsigned* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned* v = in + 6 * i;
    const uint4 r = curand_Philox4x32_10(make_uint4(v[0], v[1], v[2], v[3]), make_uint2(v[4], v[5]));
    unsigned* o = out + 8 * i;
    o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
    uint4 g = make_uint4(0, 0, 0, 0);
    if (v[1] < (1u << 30)) {
        curandStatePhilox4_32_10_t st;
        const unsigned long long seed = v[4] | (static_cast<unsigned long long>(v[5]) << 32);
        const unsigned long long subsequence = v[2] | (static_cast<unsigned long long>(v[3]) << 32);
        const unsigned long long block = v[0] | (static_cast<unsigned long long>(v[1]) << 32);
        curand_init(seed, subsequence, 4ull * block, &st);
        g = curand4(&st);
    }
    o[4] = g.x; o[5] = g.y; o[6] = g.z; o[7] = g.w;
}

extern "C" int curand_philox_blocks(int n, const unsigned* in_host, unsigned* out_host) {
    unsigned *in_dev = nullptr, *out_dev = nullptr;
    if (cudaMalloc(&in_dev, sizeof(unsigned) * 6 * n) != cudaSuccess) return -1;
    if (cudaMalloc(&out_dev, sizeof(unsigned) * 8 * n) != cudaSuccess) return -1;
    cudaMemcpy(in_dev, in_host, sizeof(unsigned) * 6 * n, cudaMemcpyHostToDevice);
    philox_blocks_kernel<<<(n + 127) / 128, 128>>>(n, in_dev, out_dev);
    const cudaError_t e = cudaMemcpy(out_host, out_dev, sizeof(unsigned) * 8 * n, cudaMemcpyDeviceToHost);
    cudaFree(in_dev);
    cudaFree(out_dev);
    return e == cudaSuccess ? 0 : -2;
}
