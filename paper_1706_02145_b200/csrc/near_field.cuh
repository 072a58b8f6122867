// near_field.cuh -- scattered electric field at arbitrary points outside the spheres, eq. (3), PAPER.md:47-49:
//
//     E_scat(r) = sum_i sum_n b^i_n Psi^(3)_n(r - r_i),
//
// with the outgoing SVWFs in their explicit form (A.2), PAPER.md:217-219 (the quantity mapped in Figs. 2 and 6,
// PAPER.md:118-120, 173-175).  One thread per field point; the spheres' coefficients and centres are staged through
// shared memory in tiles exactly as in the coupling kernel (all lanes read the same sphere).  r - r_i is formed in
// FP64, everything after it in FP32: h_l by the upward recurrence, normalised P_l^m, pi_l^m, tau_l^m (A.3) by the
// three-term recursion, the field in the local (e_r, e_theta, e_phi) frame of the pair, then rotated to Cartesian.
// O(n_points N nmax), bound by the FMA pipe.  The expansion is only valid outside sphere i (|r - r_i| > R_i).
#pragma once
#include <cuda_runtime.h>

namespace celes {

constexpr int kNearThreads = 128;
constexpr int kNearTile = 32;

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cscale(float s, float2 a) { return make_float2(s * a.x, s * a.y); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }     // i a

// kpts [n_pts][3] FP64 = k r (dimensionless, like kpos); E [n_pts][3] complex64 (x, y, z components)
template <int LMAX>
__global__ void __launch_bounds__(kNearThreads) near_field_kernel(int N, int n_pts, const double* __restrict__ kpos,
                                                                  const float2* __restrict__ b,
                                                                  const double* __restrict__ kpts, float2* __restrict__ E) {
    constexpr int H = LMAX * (LMAX + 2), NMAX = 2 * H;
    __shared__ __align__(16) float2 sb[kNearTile * NMAX];
    __shared__ double spos[kNearTile * 3];
    const int pt = blockIdx.x * kNearThreads + threadIdx.x;
    const bool active = pt < n_pts;
    const int pc = active ? pt : n_pts - 1;
    const double px = kpts[3 * (size_t)pc], py = kpts[3 * (size_t)pc + 1], pz = kpts[3 * (size_t)pc + 2];
    float2 Ex = make_float2(0.f, 0.f), Ey = Ex, Ez = Ex;
    for (int t0 = 0; t0 < N; t0 += kNearTile) {
        const int ne = min(kNearTile, N - t0);
        __syncthreads();
        {
            const float4* src = reinterpret_cast<const float4*>(b + (size_t)t0 * NMAX);
            float4* dst = reinterpret_cast<float4*>(sb);
            for (int v = threadIdx.x; v < ne * NMAX / 2; v += kNearThreads) dst[v] = __ldg(src + v);
            for (int v = threadIdx.x; v < 3 * ne; v += kNearThreads) spos[v] = kpos[(size_t)3 * t0 + v];
        }
        __syncthreads();
        for (int e = 0; e < ne; ++e) {
            const float dx = (float)(px - spos[3 * e]), dy = (float)(py - spos[3 * e + 1]), dz = (float)(pz - spos[3 * e + 2]);
            const float rho2 = fmaf(dx, dx, dy * dy), r2 = fmaf(dz, dz, rho2);
            const float rinv = rsqrtf(r2), x = r2 * rinv, ct = dz * rinv;
            const bool on_axis = rho2 < 1e-12f * r2;
            const float rhoinv = on_axis ? 0.0f : rsqrtf(rho2);
            const float cph = on_axis ? 1.0f : dx * rhoinv, sph = on_axis ? 0.0f : dy * rhoinv;
            const float st = rho2 * rhoinv * rinv;
            // h_l(x), l = 0..LMAX
            float sx, cx;
            sincos_kd(x, 0.0f, &sx, &cx);
            float2 h[LMAX + 1];
            h[0] = make_float2(sx * rinv, -cx * rinv);
            h[1] = make_float2(fmaf(sx, rinv, -cx) * rinv, -fmaf(cx, rinv, sx) * rinv);
#pragma unroll
            for (int l = 1; l < LMAX; ++l) {
                const float f = (float)(2 * l + 1) * rinv;
                h[l + 1] = make_float2(fmaf(f, h[l].x, -h[l - 1].x), fmaf(f, h[l].y, -h[l - 1].y));
            }
            // normalised P_l^m and pi_l^m = P_l^m / sin(theta) (no division: started from P_{m-1}^{m-1})
            float P[LMAX + 1][LMAX + 1], pi[LMAX + 1][LMAX + 1];
#pragma unroll
            for (int l = 0; l <= LMAX; ++l)
#pragma unroll
                for (int m = 0; m <= LMAX; ++m) { P[l][m] = 0.f; pi[l][m] = 0.f; }
            P[0][0] = 0.70710678118654752f;
#pragma unroll
            for (int m = 0; m <= LMAX; ++m) {
                if (m > 0) {
                    const float c = sqrtf((2.0f * m + 1.0f) / (2.0f * m));
                    P[m][m] = c * st * P[m - 1][m - 1];
                    pi[m][m] = c * P[m - 1][m - 1];
                }
                if (m + 1 <= LMAX) {
                    const float c = sqrtf(2.0f * m + 3.0f);
                    P[m + 1][m] = c * ct * P[m][m];
                    pi[m + 1][m] = c * ct * pi[m][m];
                }
#pragma unroll
                for (int l = m + 2; l <= LMAX; ++l) {
                    const float f1 = sqrtf((4.0f * l * l - 1.0f) / ((float)(l * l - m * m)));
                    const float f2 = sqrtf((float)((l - 1) * (l - 1) - m * m) / (4.0f * (l - 1) * (l - 1) - 1.0f));
                    P[l][m] = f1 * (ct * P[l - 1][m] - f2 * P[l - 2][m]);
                    pi[l][m] = f1 * (ct * pi[l - 1][m] - f2 * pi[l - 2][m]);
                }
            }
            float2 ph[LMAX + 1];                                   // e^{i m phi}
            ph[0] = make_float2(1.f, 0.f);
#pragma unroll
            for (int m = 1; m <= LMAX; ++m) ph[m] = cmul(ph[m - 1], make_float2(cph, sph));
            const float2* be = sb + e * NMAX;
            float2 Er = make_float2(0.f, 0.f), Et = Er, Ep = Er;   // components along e_r, e_theta, e_phi of the pair
#pragma unroll
            for (int l = 1; l <= LMAX; ++l) {
                const float nrm = rsqrtf(2.0f * l * (l + 1.0f));
                const float2 hl = h[l];
                // d(x h_l)/dx / x = h_{l-1} - l h_l / x
                const float2 dh = make_float2(fmaf(-(float)l * rinv, hl.x, h[l - 1].x), fmaf(-(float)l * rinv, hl.y, h[l - 1].y));
                const float2 hr = cscale((float)(l * (l + 1)) * rinv, hl);
#pragma unroll
                for (int m = -l; m <= l; ++m) {
                    const int am = m < 0 ? -m : m;
                    const float tau = am == 0 ? -sqrtf((float)(l * (l + 1))) * P[l][1]
                                              : l * ct * pi[l][am] - (l + am) * sqrtf((2.0f * l + 1.0f) / (2.0f * l - 1.0f) * (float)(l - am) / (float)(l + am)) * (l - 1 >= am ? pi[l - 1][am] : 0.0f);
                    const float mpi = (float)m * pi[l][am];
                    const float2 phase = m < 0 ? make_float2(ph[am].x, -ph[am].y) : ph[am];
                    const int q = (l - 1) * (l + 1) + (m + l);
                    const float2 pref = cscale(nrm, phase);
                    const float2 u = cmul(cmul(pref, be[q]), hl);          // tau = 1: pref b h_l
                    const float2 v = cmul(pref, be[H + q]);                // tau = 2: pref b
                    const float2 vd = cmul(v, dh);
                    // (A.2): Psi_1 = u (i m pi e_theta - tau e_phi);  Psi_2 = v (l(l+1) h_l / x P e_r + dh (tau e_theta + i m pi e_phi))
                    Et = cadd(Et, cadd(cscale(mpi, cmuli(u)), cscale(tau, vd)));
                    Ep = cadd(Ep, cadd(cscale(-tau, u), cscale(mpi, cmuli(vd))));
                    Er = cadd(Er, cscale(P[l][am], cmul(v, hr)));
                }
            }
            // e_r = (st cph, st sph, ct), e_theta = (ct cph, ct sph, -st), e_phi = (-sph, cph, 0)
            Ex = cadd(Ex, cadd(cadd(cscale(st * cph, Er), cscale(ct * cph, Et)), cscale(-sph, Ep)));
            Ey = cadd(Ey, cadd(cadd(cscale(st * sph, Er), cscale(ct * sph, Et)), cscale(cph, Ep)));
            Ez = cadd(Ez, cadd(cscale(ct, Er), cscale(-st, Et)));
        }
    }
    if (active) {
        E[3 * (size_t)pt] = Ex;
        E[3 * (size_t)pt + 1] = Ey;
        E[3 * (size_t)pt + 2] = Ez;
    }
}

}  // namespace celes
