// coupling_kernel.cuh -- device kernels of y = W b (steps H1-H9 of DESIGN.md section 5).
//
//   pack_kernel      b [N][nmax] -> bpm [N][nmax]: DIRECT  [b_1 + b_2 | b_1 - b_2]  (tau-block symmetry of W)
//                                                  ROTATED orthonormal [tau S|A][l][u_0,u+_1,u-_1,..] basis
//                                                  (packed variant: w_m = i u-_m in place of u-_m)
//   coupling_kernel  tiled (receiver-block x emitter-block) translation; one thread per receiver, the
//                    emitter tile (coefficients + FP64 centres) staged through shared memory, FP32 complex
//                    accumulation in registers (lmax <= 3) or in a conflict-free shared-memory slab (lmax >= 4);
//                    which (receiver block, emitter range) pieces a CTA does comes from work_partition.h
//   finalize_kernel  sums the partial-sum slots, undoes the basis transform, optional epilogue out = b - T y (eq. 9)
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
#ifdef CELES_TRACE
__device__ unsigned long long g_trace[3 * 8192];   // diagnostic builds: (smid, start ns, end ns) per CTA
#endif

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
#ifdef CELES_SLAB3
template <>
struct YPolicy<3> { using type = YSmem<nmax_of(3)>; };
#endif
template <>
struct YPolicy<4> { using type = YSmem<nmax_of(4)>; };
template <>
struct YPolicy<5> { using type = YSmem<nmax_of(5)>; };

// accumulator slab (lmax >= 4) + two emitter tiles (double buffer): coefficients [etile][nmax] and centres [etile][3]
template <int LMAX>
constexpr size_t coupling_smem_bytes(int etile) {
    return YPolicy<LMAX>::type::smem_bytes() + 2 * (size_t)etile * (nmax_of(LMAX) * sizeof(float2) + 3 * sizeof(double));
}

// Asynchronous global -> shared copies (cp.async, SASS LDGSTS): the next emitter tile is fetched while the current one
// is being translated, with no register staging and every request of the tile in flight at once.
__device__ __forceinline__ void cp_async_16(void* smem, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_8(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------------------
// grid = CTAs of the work partition (work_partition.h), cta0 + blockIdx.x is the CTA's entry in the table.  A CTA walks
// its segments: segment (rblock, [e_begin, e_end), slot) translates those emitters to receivers rblock*bs + tid,
// tid < bs, from fresh accumulators, and writes them to ypart[slot][tid][q].  Segments of receiver blocks outside
// [rb0, rb1] are skipped (row-slice calls).
//   kpos  [N][3] FP64: k * r_i.  The subtraction r_i - r_i' is done in FP64, everything after it in FP32.
template <int LMAX, int VARIANT, bool TABLE, bool EXT>
__global__ void CELES_COUPLING_BOUNDS coupling_kernel(int N, int bs, int etile, int cta0, int rb0, int rb1, HankelTable htab,
                                                          const int* __restrict__ cta_begin, const int4* __restrict__ seg,
                                                          const double* __restrict__ kpos,
                                                          const float2* __restrict__ bpm,
                                                          float2* __restrict__ ypart) {
    constexpr int NMAX = nmax_of(LMAX);
    using Y = typename YPolicy<LMAX>::type;
    extern __shared__ __align__(16) float smem_raw[];
    float* ysm = smem_raw;
    float2* sb = reinterpret_cast<float2*>(reinterpret_cast<char*>(smem_raw) + Y::smem_bytes());   // [2][etile][NMAX]
    double* spos = reinterpret_cast<double*>(sb + 2 * (size_t)etile * NMAX);                       // [2][etile][3]
    // H1: stage emitters [t0, t0 + ne) into buffer `buf` -- the coefficients are contiguous in global memory
    // (ne * NMAX float2 = ne * NMAX / 2 sixteen-byte pieces), the FP64 centres in eight-byte pieces
    auto stage = [&](int t0, int ne, int buf) {
        const float4* src = reinterpret_cast<const float4*>(bpm + (size_t)t0 * NMAX);
        float4* dst = reinterpret_cast<float4*>(sb + (size_t)buf * etile * NMAX);
        const int nvec = ne * NMAX / 2;
        for (int v = threadIdx.x; v < nvec; v += kBlock) cp_async_16(dst + v, src + v);
        double* dpos = spos + (size_t)buf * etile * 3;
        for (int v = threadIdx.x; v < 3 * ne; v += kBlock) cp_async_8(dpos + v, kpos + (size_t)3 * t0 + v);
        cp_async_commit();
    };

    const int tid = threadIdx.x;
    const int cta = cta0 + blockIdx.x;
#ifdef CELES_TRACE
    unsigned long long trace_t0 = 0;
    if (tid == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(trace_t0));
#endif
    const int s_end = cta_begin[cta + 1];
    for (int sidx = cta_begin[cta]; sidx < s_end; ++sidx) {
        const int4 sg = seg[sidx];                             // (rblock, e_begin, e_end, slot)
        if (sg.x < rb0 || sg.x > rb1) continue;
        const int i = sg.x * bs + tid;
        const bool active = tid < bs && i < N;
        const int ic = active ? i : N - 1;
        const double xi = kpos[3 * ic], yi = kpos[3 * ic + 1], zi = kpos[3 * ic + 2];

        Y yacc;
        yacc.init(ysm, tid);

        __syncthreads();                                           // the previous segment's last tile is consumed
        stage(sg.y, min(etile, sg.z - sg.y), 0);
        int buf = 0;
        for (int t0 = sg.y; t0 < sg.z; t0 += etile, buf ^= 1) {
            const int ne = min(etile, sg.z - t0);
            cp_async_wait_all();
            __syncthreads();                                       // tile t0 has landed; tile t0 - etile is consumed
            if (t0 + etile < sg.z) stage(t0 + etile, min(etile, sg.z - t0 - etile), buf ^ 1);
            const float2* tb = sb + (size_t)buf * etile * NMAX;
            const double* tp = spos + (size_t)buf * etile * 3;
            for (int e = 0; e < ne; ++e) {
                if (t0 + e == i) continue;                         // sum over i' != i (eq. 6)
                const double dx = xi - tp[3 * e];                  // d = r_i - r_i' (eq. 7), FP64 subtraction
                const double dy = yi - tp[3 * e + 1];
                const double dz = zi - tp[3 * e + 2];
                const float2* be = tb + e * NMAX;
                auto bload = [be](int q) { return be[q]; };        // same address in every lane: LDS broadcast
                pair_translate<LMAX, VARIANT, TABLE, EXT>(dx, dy, dz, htab, bload, yacc);
            }
        }
        if (active) {
            float4* dst = reinterpret_cast<float4*>(ypart + ((size_t)sg.w * kBlock + tid) * NMAX);
#pragma unroll
            for (int q = 0; q < NMAX; q += 2) {
                const float2 u = yacc.get(q), v = yacc.get(q + 1);
                dst[q / 2] = make_float4(u.x, u.y, v.x, v.y);
            }
        }
    }
#ifdef CELES_TRACE
    if (tid == 0 && blockIdx.x < 8192) {
        unsigned long long t1; unsigned smid;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        g_trace[3 * blockIdx.x] = smid; g_trace[3 * blockIdx.x + 1] = trace_t0; g_trace[3 * blockIdx.x + 2] = t1;
    }
#endif
}

// ---------------------------------------------------------------------------------------------------------
// H8-H9: for the receivers [row_begin, row_end) sums the partial-sum slots of each receiver block in slot order and
// returns to the (tau, l, m) basis; if tdiag != nullptr the epilogue of eq. (9) is fused: out = b - T y with T the
// diagonal Q^i_{tau,l} expanded to [N][nmax].  out holds rows row_begin.. only ([row_end - row_begin][nmax]); b and
// tdiag are the full [N][nmax] arrays.
//   DIRECT : y_1 = (y_+ + y_-)/2, y_2 = (y_+ - y_-)/2.
//   ROTATED: inverse of the orthonormal transform of pack_kernel.  One thread per (sphere, (l,m)).
template <int VARIANT>
__global__ void finalize_kernel(int row_begin, int row_end, int H, int bs, const int* __restrict__ slot_begin,
                                const float2* __restrict__ ypart, const float2* __restrict__ tdiag,
                                const float2* __restrict__ b, float2* __restrict__ out) {
    constexpr bool ROTATED = VARIANT != kDirect;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)(row_end - row_begin) * H) return;
    const long long i = row_begin + t / H;
    const int q = (int)(t - (i - row_begin) * H);
    const int rblock = (int)(i / bs);
    const int s0 = slot_begin[rblock], s1 = slot_begin[rblock + 1];
    const size_t stride = (size_t)kBlock * 2 * H;                  // one slot
    const float2* y0 = ypart + (size_t)(i - (long long)rblock * bs) * 2 * H;
    float2 y1, y2;
    if (!ROTATED) {
        float pr = 0.f, pi = 0.f, mr = 0.f, mi = 0.f;
        for (int s = s0; s < s1; ++s) {
            const float2 yp = y0[s * stride + q], ym = y0[s * stride + H + q];
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
        for (int s = s0; s < s1; ++s) {
            const float2* y = y0 + s * stride;
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
    const size_t r1 = o1 - (size_t)row_begin * 2 * H;
    out[r1] = y1;
    out[r1 + H] = y2;
}

}  // namespace celes
