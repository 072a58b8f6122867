// coupling_kernel.cuh -- device kernels of y = W b (steps H1-H9 of DESIGN.md section 5).
//
//   pack_kernel      b [N][nmax] -> bpm [N][nmax]: DIRECT  [b_1 + b_2 | b_1 - b_2]  (tau-block symmetry of W)
//                                                  ROTATED orthonormal [tau S|A][l][u_0,u+_1,u-_1,..] basis
//                                                  (packed variant: w_m = i u-_m in place of u-_m)
//   coupling_kernel  tiled (receiver-block x emitter-block) translation; one thread per receiver, the
//                    emitter tile (coefficients + FP64 centres) staged through shared memory, FP32 complex
//                    accumulation in registers (lmax <= 3) or in a conflict-free shared-memory slab (lmax = 4)
//   finalize_kernel  sums the emitter splits, undoes the +- transform, optional epilogue out = b - T y (eq. 9)
#pragma once
#include <cuda_runtime.h>

#include "pair_math.cuh"

namespace celes {

#ifndef CELES_KBLOCK
#define CELES_KBLOCK 128
#endif
#ifdef CELES_MAXNREG                   // tuning builds: cap the registers of the coupling kernel directly
#define CELES_COUPLING_BOUNDS __maxnreg__(CELES_MAXNREG)
#else
#define CELES_COUPLING_BOUNDS __launch_bounds__(CELES_KBLOCK)
#endif
constexpr int kBlock = CELES_KBLOCK;   // receivers (threads) per CTA

__host__ __device__ constexpr int nmax_of(int lmax) { return 2 * lmax * (lmax + 2); }

// ---------------------------------------------------------------------------------------------------------
// b -> work basis.  One thread per (sphere, index q inside a tau block).
//   DIRECT : [b_1 + b_2 | b_1 - b_2], index order unchanged.
//   ROTATED: orthonormal basis of rotation_tables.py: x_S/A = (x_1 +- x_2)/sqrt2, then per l
//            [u_0 = x_0, u+_m = (x_m + x_-m)/sqrt2, u-_m = (x_m - x_-m)/sqrt2, m = 1..l] at q = l^2-1 + {0, 2m-1, 2m}.
__device__ __forceinline__ void split_q(int q, int& l, int& pos) {
    l = 1;
    while ((l + 1) * (l + 1) - 1 <= q) ++l;
    pos = q - (l * l - 1);
}

template <int VARIANT>
__global__ void pack_kernel(int N, int H, const float2* __restrict__ b, float2* __restrict__ bpm) {
    constexpr bool ROTATED = VARIANT != kDirect;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * H) return;
    const long long i = t / H;
    const int q = (int)(t - i * H);
    const float2* b1 = b + i * 2 * H;
    const float2* b2 = b1 + H;
    float2 s, a;
    if (!ROTATED) {
        s = make_float2(b1[q].x + b2[q].x, b1[q].y + b2[q].y);
        a = make_float2(b1[q].x - b2[q].x, b1[q].y - b2[q].y);
    } else {
        int l, pos;
        split_q(q, l, pos);
        const int c0 = l * l - 1 + l;                       // index of m = 0 inside the tau block
        if (pos == 0) {
            const float r = 0.70710678118654752f;
            s = make_float2(r * (b1[c0].x + b2[c0].x), r * (b1[c0].y + b2[c0].y));
            a = make_float2(r * (b1[c0].x - b2[c0].x), r * (b1[c0].y - b2[c0].y));
        } else {
            const int m = (pos + 1) >> 1;
            const float sg = (pos & 1) ? 0.5f : -0.5f;      // u+ : x_m + x_-m ; u- : x_m - x_-m ; (1/sqrt2)^2 = 1/2
            const float2 p1 = b1[c0 + m], n1 = b1[c0 - m], p2 = b2[c0 + m], n2 = b2[c0 - m];
            const float2 u1 = make_float2(0.5f * p1.x + sg * n1.x, 0.5f * p1.y + sg * n1.y);
            const float2 u2 = make_float2(0.5f * p2.x + sg * n2.x, 0.5f * p2.y + sg * n2.y);
            s = make_float2(u1.x + u2.x, u1.y + u2.y);
            a = make_float2(u1.x - u2.x, u1.y - u2.y);
            if (!(pos & 1)) {                               // packed body: w_m = i u-_m
                s = make_float2(-s.y, s.x);
                a = make_float2(-a.y, a.x);
            }
        }
    }
    bpm[i * 2 * H + q] = s;
    bpm[i * 2 * H + H + q] = a;
}

// ---------------------------------------------------------------------------------------------------------
// Accumulator policies for y_pm of one receiver.
template <int NMAX>
struct YRegs {                       // registers: every index is a literal after unrolling
    float2 y[NMAX];
    __device__ __forceinline__ void init(float*, int) {
#pragma unroll
        for (int q = 0; q < NMAX; ++q) y[q] = make_float2(0.0f, 0.0f);
    }
    __device__ __forceinline__ void operator()(int q, float r, float i) { y[q].x += r; y[q].y += i; }
    __device__ __forceinline__ float2 get(int q) const { return y[q]; }
    __device__ __forceinline__ void put(int q, float2 v) { y[q] = v; }
    __host__ __device__ static constexpr size_t smem_bytes() { return 0; }
};

template <int NMAX>
struct YSmem {                       // shared memory slab [q][thread] (float2): lane-contiguous, conflict-free
    float2* base;
    __device__ __forceinline__ void init(float* smem, int tid) {
        base = reinterpret_cast<float2*>(smem) + tid;
#pragma unroll
        for (int q = 0; q < NMAX; ++q) base[q * kBlock] = make_float2(0.0f, 0.0f);
    }
    __device__ __forceinline__ void operator()(int q, float r, float i) {
        float2 v = base[q * kBlock];
        v.x += r; v.y += i;
        base[q * kBlock] = v;
    }
    __device__ __forceinline__ float2 get(int q) const { return base[q * kBlock]; }
    __device__ __forceinline__ void put(int q, float2 v) { base[q * kBlock] = v; }
    __host__ __device__ static constexpr size_t smem_bytes() { return sizeof(float2) * NMAX * kBlock; }
};

template <int LMAX>
struct YPolicy { using type = YRegs<nmax_of(LMAX)>; };
template <>
struct YPolicy<4> { using type = YSmem<nmax_of(4)>; };
template <>
struct YPolicy<5> { using type = YSmem<nmax_of(5)>; };

template <int LMAX>
constexpr size_t coupling_smem_bytes(int etile) {
    return YPolicy<LMAX>::type::smem_bytes() + (size_t)etile * (nmax_of(LMAX) * sizeof(float2) + 3 * sizeof(double));
}

// ---------------------------------------------------------------------------------------------------------
// grid = (ceil(N / kBlock), splits).  CTA (bx, by) translates emitters [by*chunk, min(N, (by+1)*chunk)) to
// receivers bx*kBlock + tid and writes its partial sums to ypart[by][receiver][q].
//   kpos  [N][3] FP64: k * r_i.  The subtraction r_i - r_i' is done in FP64, everything after it in FP32.
template <int LMAX, int VARIANT, bool TABLE>
__global__ void CELES_COUPLING_BOUNDS coupling_kernel(int N, int chunk, int etile, HankelTable htab,
                                                          const double* __restrict__ kpos,
                                                          const float2* __restrict__ bpm,
                                                          float2* __restrict__ ypart) {
    constexpr int NMAX = nmax_of(LMAX);
    using Y = typename YPolicy<LMAX>::type;
    extern __shared__ __align__(16) float smem_raw[];
    float* ysm = smem_raw;
    float2* sb = reinterpret_cast<float2*>(reinterpret_cast<char*>(smem_raw) + Y::smem_bytes());   // [etile][NMAX]
    double* spos = reinterpret_cast<double*>(sb + (size_t)etile * NMAX);                           // [etile][3]

    const int tid = threadIdx.x;
    const int i = blockIdx.x * kBlock + tid;
    const bool active = i < N;
    const int ic = active ? i : N - 1;
    const double xi = kpos[3 * ic], yi = kpos[3 * ic + 1], zi = kpos[3 * ic + 2];

    Y yacc;
    yacc.init(ysm, tid);

    const int e_begin = blockIdx.y * chunk;
    const int e_end = min(N, e_begin + chunk);
    for (int t0 = e_begin; t0 < e_end; t0 += etile) {
        const int ne = min(etile, e_end - t0);
        __syncthreads();                                       // previous tile fully consumed
        {   // H1: stage the tile -- coefficients are contiguous in global memory: ne * NMAX float2 = ne*NMAX/2 float4
            const float4* src = reinterpret_cast<const float4*>(bpm + (size_t)t0 * NMAX);
            float4* dst = reinterpret_cast<float4*>(sb);
            const int nvec = ne * NMAX / 2;
            for (int v = tid; v < nvec; v += kBlock) dst[v] = __ldg(src + v);
            for (int v = tid; v < 3 * ne; v += kBlock) spos[v] = kpos[(size_t)3 * t0 + v];
        }
        __syncthreads();
        for (int e = 0; e < ne; ++e) {
            if (t0 + e == i) continue;                         // sum over i' != i (eq. 6)
            const float dx = (float)(xi - spos[3 * e]);        // d = r_i - r_i' (eq. 7), FP64 subtraction
            const float dy = (float)(yi - spos[3 * e + 1]);
            const float dz = (float)(zi - spos[3 * e + 2]);
            const float2* be = sb + e * NMAX;
            auto bload = [be](int q) { return be[q]; };        // same address in every lane: LDS broadcast
            pair_translate<LMAX, VARIANT, TABLE>(dx, dy, dz, htab, bload, yacc);
        }
    }
    if (active) {
        float2* dst = ypart + ((size_t)blockIdx.y * N + i) * NMAX;
#pragma unroll
        for (int q = 0; q < NMAX; ++q) dst[q] = yacc.get(q);
    }
}

// ---------------------------------------------------------------------------------------------------------
// H8-H9: sums the emitter splits and returns to the (tau, l, m) basis; if tdiag != nullptr the epilogue of
// eq. (9) is fused: out = b - T y with T the diagonal Q^i_{tau,l} expanded to [N][nmax].
//   DIRECT : y_1 = (y_+ + y_-)/2, y_2 = (y_+ - y_-)/2.
//   ROTATED: inverse of the orthonormal transform of pack_kernel.  One thread per (sphere, (l,m)).
template <int VARIANT>
__global__ void finalize_kernel(int N, int H, int splits, const float2* __restrict__ ypart,
                                const float2* __restrict__ tdiag, const float2* __restrict__ b,
                                float2* __restrict__ out) {
    constexpr bool ROTATED = VARIANT != kDirect;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * H) return;
    const long long i = t / H;
    const int q = (int)(t - i * H);
    const size_t stride = (size_t)N * 2 * H;
    float2 y1, y2;
    if (!ROTATED) {
        float pr = 0.f, pi = 0.f, mr = 0.f, mi = 0.f;
        for (int s = 0; s < splits; ++s) {
            const float2 yp = ypart[s * stride + i * 2 * H + q], ym = ypart[s * stride + i * 2 * H + H + q];
            pr += yp.x; pi += yp.y; mr += ym.x; mi += ym.y;
        }
        y1 = make_float2(0.5f * (pr + mr), 0.5f * (pi + mi));
        y2 = make_float2(0.5f * (pr - mr), 0.5f * (pi - mi));
    } else {
        int l, pos;
        split_q(q, l, pos);
        const int m = pos - l;                               // q = l^2-1 + (m + l)
        const int base = l * l - 1;
        const int am = m < 0 ? -m : m;
        const int qa = base + (am ? 2 * am - 1 : 0);         // u+_|m| (or u_0)
        const int qb = base + 2 * am;                        // u-_|m| (unused for m = 0)
        float sar = 0.f, sai = 0.f, sbr = 0.f, sbi = 0.f, aar = 0.f, aai = 0.f, abr = 0.f, abi = 0.f;
        for (int s = 0; s < splits; ++s) {
            const float2* y = ypart + s * stride + i * 2 * H;
            const float2 sa = y[qa], aa = y[H + qa];
            sar += sa.x; sai += sa.y; aar += aa.x; aai += aa.y;
            if (am) {
                const float2 sb = y[qb], ab = y[H + qb];
                sbr += sb.x; sbi += sb.y; abr += ab.x; abi += ab.y;
            }
        }
        {                                                    // packed body: u-_m = -i w_m
            float t;
            t = sbr; sbr = sbi; sbi = -t;
            t = abr; abr = abi; abi = -t;
        }
        float ysr, ysi, yar, yai;                            // tau blocks S and A at (l, m)
        if (am == 0) { ysr = sar; ysi = sai; yar = aar; yai = aai; }
        else {
            const float r = 0.70710678118654752f, sg = m > 0 ? r : -r;
            ysr = r * sar + sg * sbr; ysi = r * sai + sg * sbi;
            yar = r * aar + sg * abr; yai = r * aai + sg * abi;
        }
        const float r = 0.70710678118654752f;
        y1 = make_float2(r * (ysr + yar), r * (ysi + yai));
        y2 = make_float2(r * (ysr - yar), r * (ysi - yai));
    }
    const size_t o1 = i * 2 * H + q, o2 = o1 + H;
    if (tdiag != nullptr) {
        const float2 t1 = tdiag[o1], t2 = tdiag[o2], b1 = b[o1], b2 = b[o2];
        y1 = make_float2(b1.x - (t1.x * y1.x - t1.y * y1.y), b1.y - (t1.x * y1.y + t1.y * y1.x));
        y2 = make_float2(b2.x - (t2.x * y2.x - t2.y * y2.y), b2.y - (t2.x * y2.y + t2.y * y2.x));
    }
    out[o1] = y1;
    out[o2] = y2;
}

}  // namespace celes
