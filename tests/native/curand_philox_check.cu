// Test infrastructure (pin P1, second half): the CUDA toolkit's own device function
// curand_Philox4x32_10(uint4 ctr, uint2 key) (curand_philox4x32_x.h) evaluated on the GPU for a list of counters.
// tests/test_gpu_parity.py compares its words with the library's device Philox (pt_philox_selftest) and with the
// oracle's.  Shares nothing with paper_2003_04621_b200/csrc or oracle/.
#include <cuda_runtime.h>
#include <curand_kernel.h>
#include <stdint.h>

__global__ void k_curand_philox(const uint4 *ctr, uint2 key, uint4 *out, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = curand_Philox4x32_10(ctr[i], key);
}

// ctr, out: HOST arrays of n x 4 uint32; returns 0 or a cudaError_t
extern "C" int curand_philox4x32_10_host(const uint32_t key[2], const uint32_t *ctr, uint32_t *out, int n)
{
    uint4 *dc = nullptr, *dout = nullptr;
    cudaError_t e = cudaMalloc(&dc, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMalloc(&dout, (size_t)n * 16);
    if (e == cudaSuccess) e = cudaMemcpy(dc, ctr, (size_t)n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_curand_philox<<<(n + 127) / 128, 128>>>(dc, make_uint2(key[0], key[1]), dout, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, (size_t)n * 16, cudaMemcpyDeviceToHost);
    cudaFree(dc);
    cudaFree(dout);
    return (int)e;
}
