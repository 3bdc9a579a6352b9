// probe.cu -- FP32 throughput probe, built into its own library (libogprobe.so), NOT part of libogtree.so:
// bench.py states the measured FP32 rate of the scalar (FFMA) and of the packed (FFMA2, fma.rn.f32x2) encoding
// next to the nominal ALU peak SMs x 128 lanes x 2 flop x clock that the roofline uses.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// 8 independent chains per thread; PACKED: each chain is a pair (two FMAs per instruction)
template <bool PACKED>
__global__ void __launch_bounds__(256) k_fp32_probe(uint64_t iters, float *sink)
{
    const float m = 0.999999f, b = 1e-7f * (float)blockIdx.x;
    float s;
    if (PACKED) {
        f32x2 a[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = pk2(threadIdx.x * 1e-3f + k, threadIdx.x * 2e-3f + k);
        const f32x2 m2 = pk2(m, m), b2 = pk2(b, b);
        for (uint64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = fma2(a[k], m2, b2);
        }
        s = 0.f;
#pragma unroll
        for (int k = 0; k < 8; ++k) s += __uint_as_float((uint32_t)a[k]) + __uint_as_float((uint32_t)(a[k] >> 32));
    } else {
        float a[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] = threadIdx.x * 1e-3f + k;
        for (uint64_t i = 0; i < iters; ++i) {
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] = fmaf(a[k], m, b);
        }
        s = 0.f;
#pragma unroll
        for (int k = 0; k < 8; ++k) s += a[k];
    }
    if (s == 123.456f) sink[0] = s;  // keeps the chains alive
}

}  // namespace

// mode 0: scalar FFMA, mode 1: packed FFMA2.  Returns 0 on success; *ms_out = device time of the timed launch
// (CUDA events on the default stream), *flops_out = flops it executed (2 per FMA).
extern "C" int ogp_fp32_probe(int mode, uint64_t iters, double *ms_out, double *flops_out)
{
    if (!ms_out || !flops_out || iters == 0 || mode < 0 || mode > 1) return -1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -4;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return -4;
    float *sink = nullptr;
    if (cudaMalloc((void **)&sink, 4096) != cudaSuccess) return -2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const unsigned grid = (unsigned)sms * 8u;
    for (int pass = 0; pass < 2; ++pass) {   // warm-up, then the timed launch
        const uint64_t n = pass == 0 ? 1000 : iters;
        if (pass == 1) cudaEventRecord(e0, 0);
        if (mode == 0) k_fp32_probe<false><<<grid, 256>>>(n, sink);
        else k_fp32_probe<true><<<grid, 256>>>(n, sink);
    }
    cudaEventRecord(e1, 0);
    int rc = 0;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = -4;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *ms_out = ms;
    *flops_out = (double)grid * 256.0 * 8.0 * (mode == 1 ? 4.0 : 2.0) * (double)iters;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    return rc;
}
