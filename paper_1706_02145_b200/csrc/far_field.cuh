// far_field.cuh -- far-field (plane-wave) amplitudes of the scattered field, PAPER.md:271 (A.12), 351-369 (D.1-D.3):
//
//     g_j(alpha, beta) = (1 / 2 pi) sum_i exp(-i k(alpha,beta).r_i) sum_n b^i_n B_nj(beta) exp(i m alpha),   j = 1, 2,
//
// "transforming [the scattered field] from the spherical wave expansion to a plane wave expansion using (A.12) for
// each of the spheres, adding up the contribution of all spheres"; I_j = 2 pi^2/(omega k mu_0) |g_j|^2.
//
//   far_field_coefficients_kernel  c[d][j][n] = B_nj(beta_d) exp(i m alpha_d) / (2 pi), B from (A.14), PAPER.md:280 (FP64)
//   far_field_kernel        device: one thread per direction (both polarisations; lmax <= 3) or per (direction,
//                           polarisation); the spheres' coefficients and k r_i are
//                           staged through shared memory in tiles (all lanes read the same sphere: broadcasts); the
//                           phase k.r_i is formed and reduced mod 2 pi in FP64 (it reaches ~1e3 rad), the rest is packed
//                           FP32 (the c_n of the thread live in registers).  O(N n_dir nmax), bound by the FMA pipe.
//                           The sphere sum is split over grid.y so that few directions still fill the device.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <vector>

namespace celes {

constexpr int kFarThreads = 128;
constexpr int kFarTile = 32;

// normalised associated Legendre functions without Condon-Shortley phase, pi = P / sin, tau = dP / d(beta)
// (A.3), 0 <= m <= l <= lmax, at one polar angle; index [l][m]
__host__ __device__ inline void legendre_pi_tau(int lmax, double ct, double st, double P[6][6], double pi[6][6], double tau[6][6]) {
    for (int l = 0; l < 6; ++l)
        for (int m = 0; m < 6; ++m) P[l][m] = pi[l][m] = tau[l][m] = 0.0;
    P[0][0] = sqrt(0.5);
    for (int m = 0; m <= lmax; ++m) {
        if (m > 0) {
            const double c = sqrt((2.0 * m + 1.0) / (2.0 * m));
            P[m][m] = c * st * P[m - 1][m - 1];
            pi[m][m] = c * P[m - 1][m - 1];                       // P_m^m / sin without dividing
        }
        if (m + 1 <= lmax) {
            P[m + 1][m] = sqrt(2.0 * m + 3.0) * ct * P[m][m];
            pi[m + 1][m] = sqrt(2.0 * m + 3.0) * ct * pi[m][m];
        }
        for (int l = m + 2; l <= lmax; ++l) {
            const double f1 = sqrt((4.0 * l * l - 1.0) / ((double)l * l - (double)m * m));
            const double f2 = sqrt((((double)l - 1.0) * (l - 1.0) - (double)m * m) / (4.0 * (l - 1.0) * (l - 1.0) - 1.0));
            P[l][m] = f1 * (ct * P[l - 1][m] - f2 * P[l - 2][m]);
            pi[l][m] = f1 * (ct * pi[l - 1][m] - f2 * pi[l - 2][m]);
        }
    }
    for (int l = 1; l <= lmax; ++l) {
        tau[l][0] = -sqrt((double)l * (l + 1.0)) * P[l][1];   // d/d(beta) P_l^0
        for (int m = 1; m <= l; ++m) {
            // sin dP_l^m/d(beta) = l cos P_l^m - (l+m) (N_lm / N_{l-1,m}) P_{l-1}^m, divided by sin through pi
            const double ratio = sqrt((2.0 * l + 1.0) / (2.0 * l - 1.0) * (double)(l - m) / (double)(l + m));
            tau[l][m] = l * ct * pi[l][m] - (l + m) * ratio * (l - 1 >= m ? pi[l - 1][m] : 0.0);
        }
    }
}

// One thread per direction: coef[(d * 2 + (j-1)) * nmax + n] = B_nj(beta_d) exp(i m alpha_d) / (2 pi) (complex64; B from
// (A.14); n in the order of celes.h) and dir[d * 3 + a] = unit vector of k(alpha_d, beta_d).  FP64.
__global__ void far_field_coefficients_kernel(int lmax, int n_dir, const double* __restrict__ alpha,
                                              const double* __restrict__ beta, float2* __restrict__ coef,
                                              double* __restrict__ dir) {
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= n_dir) return;
    const int H = lmax * (lmax + 2), nmax = 2 * H;
    double sa, ca, st, ct;
    sincos(alpha[d], &sa, &ca);
    sincos(beta[d], &st, &ct);
    dir[3 * (size_t)d] = st * ca;
    dir[3 * (size_t)d + 1] = st * sa;
    dir[3 * (size_t)d + 2] = ct;
    double P[6][6], pi[6][6], tau[6][6];
    legendre_pi_tau(lmax, ct, st, P, pi, tau);
    const double inv2pi = 0.15915494309189533577;
    for (int l = 1; l <= lmax; ++l) {
        // -1 / i^{l+1} = -(-i)^{l+1}
        double pr = 1.0, pim = 0.0;                                  // (-i)^{l+1}
        for (int t = 0; t <= l; ++t) { const double r = pim, i = -pr; pr = r; pim = i; }
        const double nrm = -inv2pi / sqrt(2.0 * l * (l + 1.0));
        const double fr = nrm * pr, fi = nrm * pim;                  // -(1/i^{l+1}) / sqrt(2l(l+1)) / 2 pi
        for (int m = -l; m <= l; ++m) {
            const int am = m < 0 ? -m : m;
            double sm, cm;
            sincos((double)m * alpha[d], &sm, &cm);
            const double er = fr * cm - fi * sm, ei = fr * sm + fi * cm;     // times exp(i m alpha)
            const int q = (l - 1) * (l + 1) + (m + l);
            for (int j = 1; j <= 2; ++j)
                for (int t = 1; t <= 2; ++t) {
                    const double ang = t == j ? tau[l][am] : m * pi[l][am];
                    // polarisation factor (i delta_j1 + delta_j2)
                    const double cr = j == 1 ? -ei * ang : er * ang, ci = j == 1 ? er * ang : ei * ang;
                    coef[((size_t)d * 2 + (j - 1)) * nmax + (t - 1) * H + q] = make_float2((float)cr, (float)ci);
                }
        }
    }
}

// grid = (ceil(n_rows / (POLS kFarThreads)), splits): CTA (x, y) sums the spheres [y * chunk, (y+1) * chunk) for its rows
// and writes gpart[y][row]; far_field_reduce_kernel adds the splits in a fixed order.  A thread owns POLS consecutive rows:
// POLS = 1, one (direction, polarisation); POLS = 2 (n_rows even), both polarisations of one direction, which share the
// FP64 phase, the sine / cosine and every shared-memory load of b (the LDS broadcast path is what limits POLS = 1:
// profiles/r02d_other_kernels.md) at twice the coefficient registers -- used while 2 NMAX complex coefficients fit.
template <int NMAX, int POLS>
__global__ void __launch_bounds__(kFarThreads) far_field_kernel(int N, int chunk, int n_rows,
                                                                const double* __restrict__ kpos,
                                                                const float2* __restrict__ b,
                                                                const float2* __restrict__ coef,
                                                                const double* __restrict__ dir, float2* __restrict__ gpart) {
    __shared__ __align__(16) float2 sb[kFarTile * NMAX];
    __shared__ double spos[kFarTile * 3];
    const int row = (blockIdx.x * kFarThreads + threadIdx.x) * POLS;   // row = direction * 2 + (j - 1)
    const bool active = row < n_rows;
    const int rc = active ? row : n_rows - POLS;
    float2 c[POLS][NMAX];
#pragma unroll
    for (int p = 0; p < POLS; ++p)
#pragma unroll
        for (int n = 0; n < NMAX; ++n) c[p][n] = coef[(size_t)(rc + p) * NMAX + n];
    const int d = rc >> 1;
    const double nx = dir[3 * d], ny = dir[3 * d + 1], nz = dir[3 * d + 2];
    float2 acc[POLS];
#pragma unroll
    for (int p = 0; p < POLS; ++p) acc[p] = make_float2(0.f, 0.f);
    const int s_begin = blockIdx.y * chunk, s_end = min(N, s_begin + chunk);
    for (int t0 = s_begin; t0 < s_end; t0 += kFarTile) {
        const int ne = min(kFarTile, s_end - t0);
        __syncthreads();
        {
            const float4* src = reinterpret_cast<const float4*>(b + (size_t)t0 * NMAX);
            float4* dst = reinterpret_cast<float4*>(sb);
            for (int v = threadIdx.x; v < ne * NMAX / 2; v += kFarThreads) dst[v] = __ldg(src + v);
            for (int v = threadIdx.x; v < 3 * ne; v += kFarThreads) spos[v] = kpos[(size_t)3 * t0 + v];
        }
        __syncthreads();
        for (int e = 0; e < ne; ++e) {
            // phase -k.r_i, reduced to [-pi, pi] in FP64
            double ph = -(nx * spos[3 * e] + ny * spos[3 * e + 1] + nz * spos[3 * e + 2]);
            ph -= 6.283185307179586476925 * rint(ph * 0.15915494309189533577);
            float sn, cs;
            __sincosf((float)ph, &sn, &cs);                         // |ph| <= pi after the FP64 reduction: hardware path
            const float4* be = reinterpret_cast<const float4*>(sb + e * NMAX);
            // sum_n c_n b_n = P + i Q per polarisation, two independent chains each
            float2 P0[POLS], Q0[POLS], P1[POLS], Q1[POLS];
#pragma unroll
            for (int p = 0; p < POLS; ++p) P0[p] = Q0[p] = P1[p] = Q1[p] = make_float2(0.f, 0.f);
#pragma unroll
            for (int n = 0; n < NMAX; n += 2) {
                const float4 bb = be[n >> 1];
                const float2 b0 = make_float2(bb.x, bb.y), b1 = make_float2(bb.z, bb.w);
#pragma unroll
                for (int p = 0; p < POLS; ++p) {
                    P0[p] = fma2(bc2(c[p][n].x), b0, P0[p]);
                    Q0[p] = fma2(bc2(c[p][n].y), b0, Q0[p]);
                    P1[p] = fma2(bc2(c[p][n + 1].x), b1, P1[p]);
                    Q1[p] = fma2(bc2(c[p][n + 1].y), b1, Q1[p]);
                }
            }
#pragma unroll
            for (int p = 0; p < POLS; ++p) {
                const float2 P = add2(P0[p], P1[p]), Q = add2(Q0[p], Q1[p]);
                const float2 s = add2(P, make_float2(-Q.y, Q.x));
                acc[p] = fma2(bc2(cs), s, acc[p]);
                acc[p] = fma2(bc2(sn), make_float2(-s.y, s.x), acc[p]);
            }
        }
    }
    if (active)
#pragma unroll
        for (int p = 0; p < POLS; ++p) gpart[(size_t)blockIdx.y * n_rows + row + p] = acc[p];
}

__global__ void far_field_reduce_kernel(int n_rows, int splits, const float2* __restrict__ gpart, float2* __restrict__ g) {
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= n_rows) return;
    float re = 0.f, im = 0.f;
    for (int s = 0; s < splits; ++s) { const float2 v = gpart[(size_t)s * n_rows + row]; re += v.x; im += v.y; }
    g[row] = make_float2(re, im);
}

}  // namespace celes
