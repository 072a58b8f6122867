// probe.cu -- FP32 throughput probes (include/celes_probe.h): measurement tools of bench.py, not part of the method.
// Built into libceles.so so that the probes run in the same process, on the same GPU, at the same clocks as the
// coupling kernel they calibrate.
#include <cuda_runtime.h>

#include <algorithm>

#include "../../include/celes.h"
#include "../../include/celes_probe.h"

#define CU_TRY(expr)                                  \
    do {                                              \
        cudaError_t e_ = (expr);                      \
        if (e_ != cudaSuccess) return e_ == cudaErrorMemoryAllocation ? CELES_ENOMEM : CELES_ECUDA; \
    } while (0)

namespace {

// ---- FP32 peak probe kernels -----------------------------------------------------------------------------
template <int VARIANT>
__global__ void __launch_bounds__(256) ffma_probe_kernel(int iters, float seed, float* sink) {
    constexpr int C = 16;                         // independent chains per thread
    float a[C];
#pragma unroll
    for (int c = 0; c < C; ++c) a[c] = seed + (float)(threadIdx.x + c);
    const float m = 0.999f + seed * 1e-9f, d = seed * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (VARIANT == 0) {
#pragma unroll
                for (int c = 0; c < C; ++c) a[c] = fmaf(a[c], m, d);
            } else if (VARIANT == 1) {
#pragma unroll
                for (int c = 0; c < C; ++c) a[c] = fmaf(a[c], 0.99951171875f, d);
            } else {
#pragma unroll
                for (int c = 0; c < C; c += 2) {
                    unsigned long long acc, mm, dd;
                    asm("mov.b64 %0, {%1, %2};" : "=l"(acc) : "f"(a[c]), "f"(a[c + 1]));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(mm) : "f"(m));
                    asm("mov.b64 %0, {%1, %1};" : "=l"(dd) : "f"(d));
                    asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc) : "l"(mm), "l"(dd));
                    asm("mov.b64 {%0, %1}, %2;" : "=f"(a[c]), "=f"(a[c + 1]) : "l"(acc));
                }
            }
        }
    }
    float t = 0.f;
#pragma unroll
    for (int c = 0; c < C; ++c) t += a[c];
    if (t == 12345.678f) sink[0] = t;             // never true in practice; keeps the chains alive
}

// Variants 3 / 4: packed fma.rn.f32x2 streams shaped like the pair body (a real coefficient times a packed complex
// value added to a packed accumulator, eight independent accumulators), in a fixed instruction order (asm
// volatile).  3: consecutive instructions share no source register (every operand is fetched from the register
// file); 4: eight consecutive instructions share the packed value (operand reuse cache).  They measure what the
// FMA pipe sustains when three register operands per instruction have to be delivered.
template <int SHARE>
__global__ void __launch_bounds__(128) ffma2_operand_probe_kernel(int iters, const float2* __restrict__ in, float* sink) {
    typedef unsigned long long u64;
    u64 R[8], z[4], u[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const float r = in[(threadIdx.x + c) & 63].x;
        asm("mov.b64 %0, {%1, %1};" : "=l"(R[c]) : "f"(r));
        asm("mov.b64 %0, {%1, %1};" : "=l"(u[c]) : "f"(0.0f));
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float2 v = in[(threadIdx.x + 8 + c) & 63];
        asm("mov.b64 %0, {%1, %2};" : "=l"(z[c]) : "f"(v.x), "f"(v.y));
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep)
#pragma unroll
            for (int m = 0; m < 4; ++m)
#pragma unroll
                for (int t = 0; t < 8; ++t) {
                    if (SHARE) asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(u[t]) : "l"(R[(t + m) & 7]), "l"(z[m]));
                    else asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(u[t]) : "l"(R[(t + m) & 7]), "l"(z[(t + m) & 3]));
                }
    }
    float acc = 0.f;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        float a, b;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(u[c]));
        acc += a + b;
    }
    if (acc == 12345.678f) sink[0] = acc;
}

}  // namespace

extern "C" {

int celes_fp32_peak_probe(int variant, int iters, double* flops_per_s, double* milliseconds, void* cuda_stream) {
    if (variant < 0 || variant > 4 || iters < 1) return CELES_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CELES_ECUDA; }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0;
    cudaDeviceProp prop;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaGetDeviceProperties(&prop, dev));
    float* sink = nullptr;
    CU_TRY(cudaMalloc(&sink, sizeof(float)));
    float2* zeros = nullptr;
    if (cudaMalloc(&zeros, 64 * sizeof(float2)) != cudaSuccess) { cudaFree(sink); return CELES_ENOMEM; }
    cudaMemsetAsync(zeros, 0, 64 * sizeof(float2), s);
    const bool operand = variant >= 3;
    const int blocks = prop.multiProcessorCount * (operand ? 4 : 8), threads = operand ? 128 : 256;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto launch = [&](int it) {
        if (variant == 0) ffma_probe_kernel<0><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 1) ffma_probe_kernel<1><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 2) ffma_probe_kernel<2><<<blocks, threads, 0, s>>>(it, 1.0f, sink);
        else if (variant == 3) ffma2_operand_probe_kernel<0><<<blocks, threads, 0, s>>>(it, zeros, sink);
        else ffma2_operand_probe_kernel<1><<<blocks, threads, 0, s>>>(it, zeros, sink);
    };
    launch(std::max(1, iters / 10));              // warm-up
    cudaEventRecord(e0, s);
    launch(iters);
    cudaEventRecord(e1, s);
    int rc = CELES_OK;
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = CELES_ECUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    cudaFree(zeros);
    const double fmas = (double)blocks * threads * (operand ? 256.0 : 128.0) * (double)iters;   // FMAs per thread and iteration
    if (flops_per_s) *flops_per_s = 2.0 * fmas / (ms * 1e-3);
    if (milliseconds) *milliseconds = ms;
    return rc;
}

}  // extern "C"
