// INT32 issue-rate microbenchmarks: the roofline denominator of the sweep kernel.
// Measures, on the bound stream with CUDA events, how many 32-bit integer thread-operations per second the
// GPU sustains for the instruction kinds the Metropolis sweep is made of.
#include "../../include/ptglass.h"
#include "../../include/ptglass_diag.h"

#include <cuda_runtime.h>
#include <stdint.h>

#include "philox.cuh"

namespace {

constexpr int ILP = 8;       // independent dependency chains per thread
constexpr int INNER = 64;    // chain steps per loop iteration

// kind 0: IMAD.WIDE.U32 only (the Philox multiply)
__global__ void mb_wide(uint32_t *out, int iters, uint32_t a)
{
    unsigned long long x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < INNER; ++j)
#pragma unroll
            for (int i = 0; i < ILP; ++i) asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(x[i]) : "r"((uint32_t)x[(i + 1) % ILP]), "r"(a));
    }
    unsigned long long s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s ^= x[i];
    if (s == 0x123456789ull) out[0] = (uint32_t)s;
}

// kind 1: LOP3 only (three-input XOR)
__global__ void mb_lop3(uint32_t *out, int iters, uint32_t a, uint32_t b)
{
    uint32_t x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < INNER; ++j)
#pragma unroll
            for (int i = 0; i < ILP; ++i) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(x[(i + 1) % ILP]), "r"(a + b));
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s ^= x[i];
    if (s == 0x12345678u) out[0] = s;
}

// kind 2: IADD3 with carry chain pair (the compare-and-pack idiom): add.cc + addc
__global__ void mb_addc(uint32_t *out, int iters, uint32_t a)
{
    uint32_t x[ILP], c[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { x[i] = threadIdx.x + i; c[i] = 0; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < INNER / 2; ++j)
#pragma unroll
            for (int i = 0; i < ILP; ++i)
                asm volatile("{ .reg .u32 t; add.cc.u32 t, %1, %2; addc.u32 %0, %0, %0; }" : "+r"(c[i]) : "r"(x[i]), "r"(a));
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s ^= c[i];
    if (s == 0x12345678u) out[0] = s;
}

// kind 3: one IMAD.WIDE + one LOP3 alternating (the Philox mix), independent chains
__global__ void mb_mix(uint32_t *out, int iters, uint32_t a, uint32_t b)
{
    unsigned long long x[ILP];
    uint32_t y[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { x[i] = threadIdx.x + i; y[i] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < INNER / 2; ++j)
#pragma unroll
            for (int i = 0; i < ILP; ++i) {
                asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(x[i]) : "r"(y[i]), "r"(a));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(y[i]) : "r"((uint32_t)(x[i] >> 32)), "r"((uint32_t)x[i]), "r"(b));
            }
    }
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s ^= y[i];
    if (s == 0x12345678u) out[0] = s;
}

// kind 4: whole Philox4x32-10 blocks, 4 independent per thread; counts 40 ops per block
__global__ void mb_philox(uint32_t *out, int iters, ptg::RoundKeys rk)
{
    uint32_t acc = 0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            uint32_t o0, o1, o2, o3;
            ptg::philox4x32_10(threadIdx.x + 1024u * i, (uint32_t)it, blockIdx.x, acc & 1u, rk, o0, o1, o2, o3);
            acc += (o0 < 0x10000000u) + (o1 < 0x10000000u) + (o2 < 0x10000000u) + (o3 < 0x10000000u);
        }
    }
    if (acc == 0xFFFFFFFFu) out[0] = acc;
}

}  // namespace

extern "C" int pt_microbench(int kind, int ctas_per_sm, int iters, void *device_scratch, void *cuda_stream,
                             double *thread_ops_per_ns, double *ms_out)
{
    if (!device_scratch || !thread_ops_per_ns || kind < 0 || kind > 4 || iters < 1 || ctas_per_sm < 1) return PT_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return PT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PT_ERR_CUDA;
    const int grid = sms * ctas_per_sm, block = 256;
    uint32_t *out = (uint32_t *)device_scratch;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double ops_per_thread = 0;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {          // first repetition is the warm-up
        cudaEventRecord(e0, st);
        switch (kind) {
        case 0: mb_wide<<<grid, block, 0, st>>>(out, iters, 0x9E3779B9u); ops_per_thread = (double)iters * INNER * ILP; break;
        case 1: mb_lop3<<<grid, block, 0, st>>>(out, iters, 0x1234567u, 0x89ABCDEu); ops_per_thread = (double)iters * INNER * ILP; break;
        case 2: mb_addc<<<grid, block, 0, st>>>(out, iters, 0x9E3779B9u); ops_per_thread = (double)iters * INNER * ILP; break;
        case 3: mb_mix<<<grid, block, 0, st>>>(out, iters, 0xD2511F53u, 0xBB67AE85u); ops_per_thread = (double)iters * INNER * ILP; break;
        case 4: mb_philox<<<grid, block, 0, st>>>(out, iters, ptg::make_round_keys(1u, 2u)); ops_per_thread = (double)iters * 4 * 40; break;
        }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) return PT_ERR_CUDA;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess) return PT_ERR_CUDA;
    *thread_ops_per_ns = ops_per_thread * (double)grid * block / ((double)best * 1e6);
    if (ms_out) *ms_out = best;
    return PT_OK;
}
