// krylov_kernels.cuh -- BLAS-1 device kernels of the host-driven GMRES loop (step H10).
// Vectors are complex64 (float2) of length n = N*nmax; every reduction accumulates in FP64.
// All scalars stay on the device between kernels (coefficients of one Gram-Schmidt pass are produced by
// dots_reduce_kernel and consumed by multi_axpy_kernel without a host round trip).
#pragma once
#include <cuda_runtime.h>

namespace celes {

constexpr int kDotBlock = 256;
constexpr int kDotChunk = 8;      // basis vectors handled per pass over w inside multi_dot_kernel

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}

// partial[block][j] = sum over this block's elements of conj(V_j[t]) * w[t],  j < k.   V_j = V + j*n.
__global__ void __launch_bounds__(kDotBlock) multi_dot_kernel(long long n, int k, const float2* __restrict__ V,
                                                              const float2* __restrict__ w,
                                                              double2* __restrict__ partial) {
    __shared__ double sre[kDotBlock / 32][kDotChunk], sim[kDotBlock / 32][kDotChunk];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j0 = 0; j0 < k; j0 += kDotChunk) {
        double ar[kDotChunk], ai[kDotChunk];
#pragma unroll
        for (int c = 0; c < kDotChunk; ++c) { ar[c] = 0.0; ai[c] = 0.0; }
        for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
            const float2 wv = w[t];
#pragma unroll
            for (int c = 0; c < kDotChunk; ++c) {
                if (j0 + c < k) {
                    const float2 v = V[(size_t)(j0 + c) * n + t];
                    ar[c] += (double)v.x * wv.x + (double)v.y * wv.y;     // conj(v) * w
                    ai[c] += (double)v.x * wv.y - (double)v.y * wv.x;
                }
            }
        }
#pragma unroll
        for (int c = 0; c < kDotChunk; ++c) {
            const double r = warp_sum(ar[c]), i = warp_sum(ai[c]);
            if (lane == 0) { sre[warp][c] = r; sim[warp][c] = i; }
        }
        __syncthreads();
        if (threadIdx.x < kDotChunk && j0 + threadIdx.x < k) {
            double r = 0.0, i = 0.0;
            for (int q = 0; q < kDotBlock / 32; ++q) { r += sre[q][threadIdx.x]; i += sim[q][threadIdx.x]; }
            partial[(size_t)blockIdx.x * k + j0 + threadIdx.x] = make_double2(r, i);
        }
        __syncthreads();
    }
}

// out[j] = sum_b partial[b][j]; if accum != nullptr also accum[j] += out[j] (CGS2: h = h1 + h2).
// One CTA of kReduceThreads per inner product j: the nblocks partial sums are read in parallel (a serial loop over
// them in one thread costs nblocks dependent L2 latencies, which dominated the Krylov overhead), summed in a fixed
// order per thread, then by warp shuffles and a shared-memory pass -- deterministic.
constexpr int kReduceThreads = 128;
__global__ void __launch_bounds__(kReduceThreads) dots_reduce_kernel(int nblocks, int k, const double2* __restrict__ partial,
                                                                     double2* __restrict__ out, double2* __restrict__ accum) {
    __shared__ double sr[kReduceThreads / 32], si[kReduceThreads / 32];
    const int j = blockIdx.x;
    if (j >= k) return;
    double r = 0.0, i = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += kReduceThreads) { const double2 p = partial[(size_t)b * k + j]; r += p.x; i += p.y; }
    r = warp_sum(r); i = warp_sum(i);
    if ((threadIdx.x & 31) == 0) { sr[threadIdx.x >> 5] = r; si[threadIdx.x >> 5] = i; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tr = 0.0, ti = 0.0;
        for (int q = 0; q < kReduceThreads / 32; ++q) { tr += sr[q]; ti += si[q]; }
        out[j] = make_double2(tr, ti);
        if (accum != nullptr) { accum[j].x += tr; accum[j].y += ti; }
    }
}

// w[t] += alpha * sum_{j<k} coef[j] * V_j[t]       (alpha = -1: orthogonalisation, +1: solution update)
__global__ void multi_axpy_kernel(long long n, int k, double alpha, const double2* __restrict__ coef,
                                  const float2* __restrict__ V, float2* __restrict__ w) {
    extern __shared__ double2 sc[];
    for (int j = threadIdx.x; j < k; j += blockDim.x) sc[j] = make_double2(alpha * coef[j].x, alpha * coef[j].y);
    __syncthreads();
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const float2 w0 = w[t];
        double r = w0.x, i = w0.y;
        for (int j = 0; j < k; ++j) {
            const float2 v = V[(size_t)j * n + t];
            r += sc[j].x * v.x - sc[j].y * v.y;
            i += sc[j].x * v.y + sc[j].y * v.x;
        }
        w[t] = make_float2((float)r, (float)i);
    }
}

// out = w / sqrt(nrm2[0].x)   (nrm2 = <w,w> from the dot kernels); out may alias w (so neither is __restrict__)
__global__ void scale_by_inv_norm_kernel(long long n, const double2* __restrict__ nrm2, const float2* w, float2* out) {
    const double s = nrm2[0].x > 0.0 ? rsqrt(nrm2[0].x) : 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const float2 v = w[t];
        out[t] = make_float2((float)(v.x * s), (float)(v.y * s));
    }
}

// out = a - b
__global__ void sub_kernel(long long n, const float2* __restrict__ a, const float2* __restrict__ b, float2* __restrict__ out) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        out[t] = make_float2(a[t].x - b[t].x, a[t].y - b[t].y);
}

// out = a x + b y + c z  (complex scalars by value; y, z may be nullptr when their scalar is unused; out may alias
// any input).  The vector updates of BiCGSTAB.
__global__ void lincomb_kernel(long long n, double2 a, const float2* x, double2 b, const float2* y, double2 c,
                               const float2* z, float2* out) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
        const float2 xv = x[t];
        double r = a.x * xv.x - a.y * xv.y, i = a.x * xv.y + a.y * xv.x;
        if (y != nullptr) { const float2 v = y[t]; r += b.x * v.x - b.y * v.y; i += b.x * v.y + b.y * v.x; }
        if (z != nullptr) { const float2 v = z[t]; r += c.x * v.x - c.y * v.y; i += c.x * v.y + c.y * v.x; }
        out[t] = make_float2((float)r, (float)i);
    }
}

// out = T a (diagonal), used for the right-hand side of eq. (8)
__global__ void tapply_kernel(long long n, const float2* __restrict__ tdiag, const float2* __restrict__ a,
                              float2* __restrict__ out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const float2 q = tdiag[t], v = a[t];
    out[t] = make_float2(q.x * v.x - q.y * v.y, q.x * v.y + q.y * v.x);
}

// x += y
__global__ void add_kernel(long long n, const float2* __restrict__ y, float2* __restrict__ x) {
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x)
        x[t] = make_float2(x[t].x + y[t].x, x[t].y + y[t].y);
}

}  // namespace celes
