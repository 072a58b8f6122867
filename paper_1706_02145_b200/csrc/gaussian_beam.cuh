// gaussian_beam.cuh -- initial-field coefficients of the Gaussian beam of Appendix C, (C.8) with (C.7),
// PAPER.md:302-348:
//
//   a^i_{in,n} = E0 k^2 w^2 / pi  sum_j int_0^{pi/2} d(beta) sin(beta) cos(beta) B^dagger_nj(beta) I_jn(beta)
//                exp[-w^2 k^2 sin^2(beta) / 4 + i k z_Gi cos(beta)],
//   I_jn = 2 pi e^{-i aG} i^{|m-1|} e^{-i(m-1) phi_Gi} J_{|m-1|}(k rho_Gi sin(beta)) (d_j1 - i d_j2)/2
//        + 2 pi e^{+i aG} i^{|m+1|} e^{-i(m+1) phi_Gi} J_{|m+1|}(k rho_Gi sin(beta)) (d_j1 + i d_j2)/2,
//
// (rho, phi, z)_Gi the cylindrical coordinates of r_i - r_G.  O(N nmax n_beta) input preparation, done in FP64 and
// rounded once to complex64.  The beta-integral uses Gauss-Legendre nodes on [0, pi/2] (host: nodes, weights and the
// sphere-independent factor  wgt_q B^dagger_nj(beta_q) (d_j1 -+ i d_j2)/2  summed over j; device: the rest).
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <vector>

#include "far_field.cuh"   // legendre_pi_tau

namespace celes {

// Gauss-Legendre nodes / weights on [-1, 1] by Newton iteration on P_n
inline void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
    x.resize(n); w.resize(n);
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = std::cos(M_PI * (i + 0.75) / (n + 0.5)), pp = 0.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            const double dz = p1 / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-15) break;
        }
        x[i] = -z; x[n - 1 - i] = z;
        w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

// Host tables of the quadrature: sb[q], cb[q] = sin, cos(beta_q);
// cminus[q][n] = wgt_q sum_j B^dagger_nj (d_j1 - i d_j2)/2,  cplus[q][n] = wgt_q sum_j B^dagger_nj (d_j1 + i d_j2)/2,
// wgt_q = GL weight x sin cos exp(-w^2 k^2 sin^2 / 4) x 2 pi x k^2 w^2 / pi   (everything that does not depend on the sphere)
inline void gaussian_beam_tables(int lmax, int n_beta, double k, double w, std::vector<double>& sb, std::vector<double>& cb,
                                 std::vector<double2>& cminus, std::vector<double2>& cplus) {
    const int H = lmax * (lmax + 2), nmax = 2 * H;
    std::vector<double> x, wq;
    gauss_legendre(n_beta, x, wq);
    sb.resize(n_beta); cb.resize(n_beta);
    cminus.assign((size_t)n_beta * nmax, make_double2(0.0, 0.0));
    cplus.assign((size_t)n_beta * nmax, make_double2(0.0, 0.0));
    typedef std::complex<double> cd;
    const cd I(0.0, 1.0);
    for (int q = 0; q < n_beta; ++q) {
        const double beta = (x[q] + 1.0) * M_PI / 4.0;
        sb[q] = std::sin(beta); cb[q] = std::cos(beta);
        const double wgt = wq[q] * M_PI / 4.0 * sb[q] * cb[q] * std::exp(-w * w * k * k * sb[q] * sb[q] / 4.0) * 2.0 * k * k * w * w;
        double P[6][6], pi[6][6], tau[6][6];
        legendre_pi_tau(lmax, cb[q], sb[q], P, pi, tau);
        for (int t = 1; t <= 2; ++t)
            for (int l = 1; l <= lmax; ++l)
                for (int m = -l; m <= l; ++m) {
                    const int am = m < 0 ? -m : m;
                    cd bd[3];
                    for (int j = 1; j <= 2; ++j) {
                        const double ang = t == j ? tau[l][am] : m * pi[l][am];
                        // (A.14) with every explicit i -> -i
                        bd[j] = -1.0 / std::pow(-I, l + 1) / std::sqrt(2.0 * l * (l + 1.0)) * (j == 1 ? -I : cd(1.0)) * ang;
                    }
                    const cd cm = wgt * (bd[1] - I * bd[2]) / 2.0, cp = wgt * (bd[1] + I * bd[2]) / 2.0;
                    const size_t o = (size_t)q * nmax + (t - 1) * H + (l - 1) * (l + 1) + (m + l);
                    cminus[o] = make_double2(cm.real(), cm.imag());
                    cplus[o] = make_double2(cp.real(), cp.imag());
                }
    }
}

// One thread per (sphere, n).  kpos = k r_i (FP64), krG = k r_G.
__global__ void gaussian_beam_kernel(int N, int lmax, int n_beta, const double* __restrict__ kpos, double krGx, double krGy,
                                     double krGz, double alpha_G, double2 E0, const double* __restrict__ sb,
                                     const double* __restrict__ cb, const double2* __restrict__ cminus,
                                     const double2* __restrict__ cplus, float2* __restrict__ a_in) {
    const int H = lmax * (lmax + 2), nmax = 2 * H;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * nmax) return;
    const int i = (int)(t / nmax), n = (int)(t - (long long)i * nmax);
    const int qn = n % H;
    int l = 1;
    while ((l + 1) * (l + 1) - 1 <= qn) ++l;
    const int m = qn - (l * l - 1) - l;
    const double dx = kpos[3 * i] - krGx, dy = kpos[3 * i + 1] - krGy, kz = kpos[3 * i + 2] - krGz;
    const double krho = sqrt(dx * dx + dy * dy), phi = atan2(dy, dx);
    const int m1 = m - 1, m2 = m + 1, n1 = m1 < 0 ? -m1 : m1, n2 = m2 < 0 ? -m2 : m2;
    // e^{-+ i aG} i^{|m -+ 1|} e^{-i (m -+ 1) phi}
    double s1, c1, s2, c2;
    sincos(-alpha_G - m1 * phi + 1.5707963267948966 * n1, &s1, &c1);
    sincos(alpha_G - m2 * phi + 1.5707963267948966 * n2, &s2, &c2);
    double ar = 0.0, ai = 0.0;
    for (int q = 0; q < n_beta; ++q) {
        const double x = krho * sb[q];
        const double j1 = jn(n1, x), j2 = jn(n2, x);
        const double2 cm = cminus[(size_t)q * nmax + n], cp = cplus[(size_t)q * nmax + n];
        // term = cm e1 J1 + cp e2 J2, e1 = (c1, s1), e2 = (c2, s2)
        const double tr = (cm.x * c1 - cm.y * s1) * j1 + (cp.x * c2 - cp.y * s2) * j2;
        const double ti = (cm.x * s1 + cm.y * c1) * j1 + (cp.x * s2 + cp.y * c2) * j2;
        double sz, cz;
        sincos(kz * cb[q], &sz, &cz);                                  // e^{i k z_Gi cos(beta)}
        ar += tr * cz - ti * sz;
        ai += tr * sz + ti * cz;
    }
    a_in[t] = make_float2((float)(E0.x * ar - E0.y * ai), (float)(E0.x * ai + E0.y * ar));
}

// Plane wave E0 Phi_j(alpha, beta; r) expanded about every sphere centre, (A.13)-(A.14), PAPER.md:276-282:
//   a^i_{in,n} = E0 exp(i k.r_i) 4 exp(-i m alpha) B^dagger_nj(beta).   One thread per (sphere, n), FP64, rounded once.
__global__ void plane_wave_kernel(int N, int lmax, const double* __restrict__ kpos, double alpha, double beta, int j,
                                  double2 E0, float2* __restrict__ a_in) {
    const int H = lmax * (lmax + 2), nmax = 2 * H;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)N * nmax) return;
    const int i = (int)(t / nmax), n = (int)(t - (long long)i * nmax);
    const int tau = n / H + 1, qn = n % H;
    int l = 1;
    while ((l + 1) * (l + 1) - 1 <= qn) ++l;
    const int m = qn - (l * l - 1) - l, am = m < 0 ? -m : m;
    double sa, ca, sb, cb;
    sincos(alpha, &sa, &ca);
    sincos(beta, &sb, &cb);
    double P[6][6], pi[6][6], tt[6][6];
    legendre_pi_tau(lmax, cb, sb, P, pi, tt);
    const double ang = tau == j ? tt[l][am] : m * pi[l][am];
    // B^dagger_nj = -(1 / (-i)^{l+1}) / sqrt(2 l (l+1)) (-i d_j1 + d_j2) ang;   1 / (-i)^{l+1} = i^{l+1}
    double pr = 1.0, pim = 0.0;                                      // i^{l+1}
    for (int q = 0; q <= l; ++q) { const double r = -pim, im = pr; pr = r; pim = im; }
    const double nrm = -4.0 * ang / sqrt(2.0 * l * (l + 1.0));
    double br = nrm * pr, bi = nrm * pim;
    if (j == 1) { const double r = bi, im = -br; br = r; bi = im; }    // times -i
    // phase exp(i (k.r_i - m alpha))
    const double ph = (sb * ca) * kpos[3 * i] + (sb * sa) * kpos[3 * i + 1] + cb * kpos[3 * i + 2] - m * alpha;
    double sp, cp;
    sincos(ph, &sp, &cp);
    const double vr = br * cp - bi * sp, vi = br * sp + bi * cp;
    a_in[t] = make_float2((float)(E0.x * vr - E0.y * vi), (float)(E0.x * vi + E0.y * vr));
}

}  // namespace celes
