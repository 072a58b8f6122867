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
            h[0] = mul2(bc2(rinv), make_float2(sx, -cx));
            h[1] = fma2(bc2(rinv), h[0], nimul2(h[0]));             // h_1 = h_0 / x - e^{ix} / x,  e^{ix} / x = i h_0
#pragma unroll
            for (int l = 1; l < LMAX; ++l) h[l + 1] = fma2(bc2((float)(2 * l + 1) * rinv), h[l], neg2(h[l - 1]));
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
            for (int m = 1; m <= LMAX; ++m) ph[m] = cmul2(make_float2(cph, sph), ph[m - 1]);
            const float2* be = sb + e * NMAX;
            float2 Er = make_float2(0.f, 0.f), Et = Er, Ep = Er;   // components along e_r, e_theta, e_phi of the pair
            // (A.2): Psi_1 = u (i m pi e_theta - tau e_phi),  Psi_2 = v (l(l+1) h_l / x P e_r + dh (tau e_theta + i m pi e_phi)),
            // u = nrm e^{i m phi} b_1 h_l, v = nrm e^{i m phi} b_2.  The radial factors depend on l only: the five angular sums
            // over m are formed first (packed: one FFMA2 per real coefficient x complex value) and meet h_l, dh, h_l / x once per l.
#pragma unroll
            for (int l = 1; l <= LMAX; ++l) {
                const float nrm = rsqrtf(2.0f * l * (l + 1.0f));
                const float2 hl = h[l];
                // d(x h_l)/dx / x = h_{l-1} - l h_l / x
                const float2 dh = fma2(bc2(-(float)l * rinv), hl, h[l - 1]);
                const float2 hlN = mul2(bc2(nrm), hl), dhN = mul2(bc2(nrm), dh), hrN = mul2(bc2(nrm * (float)(l * (l + 1)) * rinv), hl);
                float2 S1 = make_float2(0.f, 0.f), S2 = S1, T1 = S1, T2 = S1, T3 = S1;
#pragma unroll
                for (int m = -l; m <= l; ++m) {
                    const int am = m < 0 ? -m : m;
                    const float tau = am == 0 ? -sqrtf((float)(l * (l + 1))) * P[l][1]
                                              : l * ct * pi[l][am] - (l + am) * sqrtf((2.0f * l + 1.0f) / (2.0f * l - 1.0f) * (float)(l - am) / (float)(l + am)) * (l - 1 >= am ? pi[l - 1][am] : 0.0f);
                    const float2 phase = m < 0 ? make_float2(ph[am].x, -ph[am].y) : ph[am];
                    const int q = (l - 1) * (l + 1) + (m + l);
                    const float2 c1 = m == 0 ? be[q] : cmul2(phase, be[q]);           // e^{i m phi} b_1
                    const float2 c2 = m == 0 ? be[H + q] : cmul2(phase, be[H + q]);   // e^{i m phi} b_2
                    S2 = fma2(bc2(-tau), c1, S2);
                    T1 = fma2(bc2(tau), c2, T1);
                    T3 = fma2(bc2(P[l][am]), c2, T3);
                    if (m != 0) {
                        const float mpi = (float)m * pi[l][am];
                        S1 = fma2(bc2(mpi), imul2(c1), S1);
                        T2 = fma2(bc2(mpi), imul2(c2), T2);
                    }
                }
                Et = cfma2(dhN, T1, cfma2(hlN, S1, Et));
                Ep = cfma2(dhN, T2, cfma2(hlN, S2, Ep));
                Er = cfma2(hrN, T3, Er);
            }
            // e_r = (st cph, st sph, ct), e_theta = (ct cph, ct sph, -st), e_phi = (-sph, cph, 0)
            Ex = fma2(bc2(-sph), Ep, fma2(bc2(ct * cph), Et, fma2(bc2(st * cph), Er, Ex)));
            Ey = fma2(bc2(cph), Ep, fma2(bc2(ct * sph), Et, fma2(bc2(st * sph), Er, Ey)));
            Ez = fma2(bc2(-st), Et, fma2(bc2(ct), Er, Ez));
        }
    }
    if (active) {
        E[3 * (size_t)pt] = Ex;
        E[3 * (size_t)pt + 1] = Ey;
        E[3 * (size_t)pt + 2] = Ez;
    }
}

}  // namespace celes
