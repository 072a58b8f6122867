// =============================================================================
// CELES oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain double-precision CPU restatement of the coupling operator of
// arxiv 1706.02145, written from the paper's equations only:
//   * eq. (6)-(7)   a^i_n = a_in + sum_{i'!=i} sum_{n'} W^{ii'}_{nn'} b^{i'}_{n'},
//                                      W^{ii'}_{nn'} = A_{n'n}(r_i - r_i')
//   * eq. (A.6)-(A.8) closed-form translation operator
//   * eq. (A.9)-(A.11) a5 / b5 coefficients with Wigner-3j symbols
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.  It shares no code, header, table or constant with the
// CUDA path under paper_1706_02145_b200/ and neither includes the other.
//
// Special functions come from the C++17 <cmath> library (std::sph_bessel,
// std::sph_neumann, std::assoc_legendre -- the latter has NO Condon-Shortley phase),
// the Wigner-3j symbol from the Racah single-sum formula written out below.
// There is no blocking, fusion or reordering beyond caching the a5/b5 table (they do
// not depend on the pair) and the per-pair h_p, P_p^mu values.
//
// Readings of the paper used here are DESIGN.md R1-R8 (index order, normalisation of
// P_l^m, direction of d, sign of the azimuthal phase, phi on the z axis).
//
// Pins (tests/test_oracle_pins.py): brute-force addition theorem (A.5), physical form
// of eq. (7), on-axis m-diagonality, d -> -d parity, tau-block structure, golden W
// entries, Wigner-3j orthogonality and exact SymPy values.  Nothing here is unpinned.
// =============================================================================
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

// ---------------------------------------------------------------- factorials
static long double factorial_ld(int n) {
    long double f = 1.0L;
    for (int i = 2; i <= n; ++i) f *= (long double)i;
    return f;
}

// ---------------------------------------------------------------- Wigner 3j
// Racah formula.  ( j1 j2 j3 ; m1 m2 m3 ), integer arguments only.
static double wigner3j(int j1, int j2, int j3, int m1, int m2, int m3) {
    if (j1 < 0 || j2 < 0 || j3 < 0) return 0.0;
    if (m1 + m2 + m3 != 0) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m3) > j3) return 0.0;
    if (j3 > j1 + j2 || j3 < std::abs(j1 - j2)) return 0.0;
    long double delta = factorial_ld(j1 + j2 - j3) * factorial_ld(j1 - j2 + j3) *
                        factorial_ld(-j1 + j2 + j3) / factorial_ld(j1 + j2 + j3 + 1);
    long double pref = sqrtl(delta * factorial_ld(j1 + m1) * factorial_ld(j1 - m1) *
                             factorial_ld(j2 + m2) * factorial_ld(j2 - m2) *
                             factorial_ld(j3 + m3) * factorial_ld(j3 - m3));
    long double sum = 0.0L;
    for (int t = 0; t <= j1 + j2 + j3; ++t) {
        int d1 = j3 - j2 + t + m1, d2 = j3 - j1 + t - m2, d3 = j1 + j2 - j3 - t;
        int d4 = j1 - t - m1, d5 = j2 - t + m2;
        if (d1 < 0 || d2 < 0 || d3 < 0 || d4 < 0 || d5 < 0) continue;
        long double den = factorial_ld(t) * factorial_ld(d1) * factorial_ld(d2) *
                          factorial_ld(d3) * factorial_ld(d4) * factorial_ld(d5);
        sum += ((t & 1) ? -1.0L : 1.0L) / den;
    }
    int ph = j1 - j2 - m3;
    long double sgn = (ph & 1) ? -1.0L : 1.0L;   // (ph & 1) is right for negative ph too
    return (double)(sgn * pref * sum);
}

// i^k for any integer k
static cplx ipow(int k) {
    int r = ((k % 4) + 4) % 4;
    switch (r) {
        case 0: return cplx(1, 0);
        case 1: return cplx(0, 1);
        case 2: return cplx(-1, 0);
        default: return cplx(0, -1);
    }
}

// ---------------------------------------------------------------- a5, b5 (A.9)-(A.11)
static cplx a5(int l, int m, int lp, int mp, int p) {
    cplx phase = ipow(std::abs(m - mp) - std::abs(m) - std::abs(mp) + lp - l + p) *
                 (((m - mp) & 1) ? -1.0 : 1.0);
    double f = (double)(l * (l + 1) + lp * (lp + 1) - p * (p + 1)) * std::sqrt(2.0 * p + 1.0) *
               std::sqrt((2.0 * l + 1.0) * (2.0 * lp + 1.0) / (2.0 * l * (l + 1.0) * lp * (lp + 1.0)));
    return phase * f * wigner3j(l, lp, p, m, -mp, mp - m) * wigner3j(l, lp, p, 0, 0, 0);
}

static cplx b5(int l, int m, int lp, int mp, int p) {
    cplx phase = ipow(std::abs(m - mp) - std::abs(m) - std::abs(mp) + lp - l + p) *
                 (((m - mp) & 1) ? -1.0 : 1.0);
    double rad = (double)(l + lp + 1 + p) * (double)(l + lp + 1 - p) * (double)(p + l - lp) *
                 (double)(p - l + lp) * (2.0 * p + 1.0);
    if (rad < 0.0) return cplx(0, 0);
    double f = std::sqrt(rad) *
               std::sqrt((2.0 * lp + 1.0) * (2.0 * l + 1.0) / (2.0 * l * (l + 1.0) * lp * (lp + 1.0)));
    return phase * f * wigner3j(l, lp, p, m, -mp, mp - m) * wigner3j(l, lp, p - 1, 0, 0, 0);
}

// ---------------------------------------------------------------- special functions
// normalised associated Legendre function, reading R2:
//   P_l^m(x) = sqrt((2l+1)/2 (l-m)!/(l+m)!) (1-x^2)^{m/2} d^m/dx^m P_l(x),  0 <= m <= l
static double legendre_normalized(int l, int m, double x) {
    if (m < 0 || m > l) return 0.0;
    long double nrm = sqrtl((2.0L * l + 1.0L) / 2.0L * factorial_ld(l - m) / factorial_ld(l + m));
    return (double)nrm * std::assoc_legendre((unsigned)l, (unsigned)m, x);
}

// radial function z_p(x): kind 3 -> h_p^(1) = j_p + i y_p, kind 1 -> j_p, kind 2 -> y_p.
// libstdc++'s std::sph_bessel refuses arguments beyond about 1.5e4 ("Argument x too large in __bessel_jn") and has
// lost six digits by 1e4; for x > kLargeArgument the textbook closed forms j_0 = sin x / x, j_1 = sin x / x^2 - cos x / x,
// y_0 = -cos x / x, y_1 = -cos x / x^2 - sin x / x and the three-term recurrence f_{p+1} = (2p+1)/x f_p - f_{p-1}
// are used instead (upward recurrence is stable for x >> p; p <= 2 lmax <= 10 here).  Pinned against SciPy / mpmath on
// both sides of the switch (tests/test_oracle_pins.py::test_radial_large_argument).
static const double kLargeArgument = 8000.0;
static cplx radial(int kind, int p, double x) {
    double j, y;
    if (x > kLargeArgument) {
        const double s = std::sin(x), c = std::cos(x);
        double j0 = s / x, j1 = s / (x * x) - c / x, y0 = -c / x, y1 = -c / (x * x) - s / x;
        if (p == 0) { j = j0; y = y0; }
        else {
            for (int q = 1; q < p; ++q) {
                const double jn = (2.0 * q + 1.0) / x * j1 - j0, yn = (2.0 * q + 1.0) / x * y1 - y0;
                j0 = j1; j1 = jn; y0 = y1; y1 = yn;
            }
            j = j1; y = y1;
        }
    } else {
        j = kind == 2 ? 0.0 : std::sph_bessel((unsigned)p, x);
        y = kind == 1 ? 0.0 : std::sph_neumann((unsigned)p, x);
    }
    if (kind == 1) return cplx(j, 0.0);
    if (kind == 2) return cplx(y, 0.0);
    return cplx(j, y);
}

// spherical coordinates of d; phi := 0 on the z axis (reading R8)
static void spherical(double dx, double dy, double dz, double* d, double* ct, double* phi) {
    *d = std::sqrt(dx * dx + dy * dy + dz * dz);
    *ct = dz / *d;
    *phi = (dx == 0.0 && dy == 0.0) ? 0.0 : std::atan2(dy, dx);
}

// ---------------------------------------------------------------- A_{nn'}(d), (A.6)-(A.8)
// n = (tau,l,m), n' = (tau',l',m').  The "p,p'" of (A.6) are tau,tau' (reading R4).
static cplx translation_A(int tau, int l, int m, int taup, int lp, int mp, double k,
                          double dx, double dy, double dz, int kind) {
    double d, ct, phi;
    spherical(dx, dy, dz, &d, &ct, &phi);
    int mu = std::abs(m - mp);
    cplx sum(0, 0);
    if (tau == taup) {
        for (int p = std::abs(l - lp); p <= l + lp; ++p)
            sum += a5(l, m, lp, mp, p) * radial(kind, p, k * d) * legendre_normalized(p, mu, ct);
    } else {
        for (int p = std::abs(l - lp) + 1; p <= l + lp; ++p)
            sum += b5(l, m, lp, mp, p) * radial(kind, p, k * d) * legendre_normalized(p, mu, ct);
    }
    return std::exp(cplx(0, (m - mp) * phi)) * sum;
}

// multi-index (reading R1): n = (tau-1) nmax/2 + (l-1)(l+1) + (m+l), 0-based
static inline int nindex(int lmax, int tau, int l, int m) {
    return (tau - 1) * lmax * (lmax + 2) + (l - 1) * (l + 1) + (m + l);
}

// ---------------------------------------------------------------- cached coefficient table
// a5/b5 do not depend on the pair: evaluate the functions above once per call
// and reuse the values.  table index [l][m+l][l'][m'+l'][p], p = 0..2 lmax.
struct CoefTable {
    int lmax, P;
    std::vector<cplx> a, b;
    size_t idx(int l, int m, int lp, int mp, int p) const {
        int L = lmax + 1, M = 2 * lmax + 1;
        return ((((size_t)l * M + (m + l)) * L + lp) * M + (mp + lp)) * P + p;
    }
    explicit CoefTable(int lmax_) : lmax(lmax_), P(2 * lmax_ + 1) {
        int L = lmax + 1, M = 2 * lmax + 1;
        a.assign((size_t)L * M * L * M * P, cplx(0, 0));
        b.assign((size_t)L * M * L * M * P, cplx(0, 0));
        for (int l = 1; l <= lmax; ++l) for (int m = -l; m <= l; ++m)
        for (int lp = 1; lp <= lmax; ++lp) for (int mp = -lp; mp <= lp; ++mp) {
            for (int p = std::abs(l - lp); p <= l + lp; ++p) a[idx(l, m, lp, mp, p)] = a5(l, m, lp, mp, p);
            for (int p = std::abs(l - lp) + 1; p <= l + lp; ++p) b[idx(l, m, lp, mp, p)] = b5(l, m, lp, mp, p);
        }
    }
};

// W^{ii'} block for d = r_i - r_i' (eq. 7): W[n][n'] = A_{n'n}(d), row-major nmax x nmax
static void coupling_block(const CoefTable& T, double k, double dx, double dy, double dz, int kind, cplx* W) {
    const int lmax = T.lmax, P = T.P;
    double d, ct, phi;
    spherical(dx, dy, dz, &d, &ct, &phi);
    std::vector<cplx> z(P);
    std::vector<double> leg((size_t)P * P, 0.0);   // leg[p*P + mu]
    for (int p = 0; p < P; ++p) {
        z[p] = radial(kind, p, k * d);
        for (int mu = 0; mu <= p; ++mu) leg[(size_t)p * P + mu] = legendre_normalized(p, mu, ct);
    }
    std::vector<cplx> phase(2 * P - 1);            // phase[mu + 2 lmax] = e^{i mu phi}, mu = m' - m
    for (int mu = -(P - 1); mu <= P - 1; ++mu) phase[mu + P - 1] = std::exp(cplx(0, mu * phi));
    const int nmax = 2 * lmax * (lmax + 2);
    for (int tau = 1; tau <= 2; ++tau) for (int l = 1; l <= lmax; ++l) for (int m = -l; m <= l; ++m)      // receiver n
    for (int taup = 1; taup <= 2; ++taup) for (int lp = 1; lp <= lmax; ++lp) for (int mp = -lp; mp <= lp; ++mp) {  // emitter n'
        // W_{nn'} = A_{n'n}: first index of A is the emitter n', second the receiver n
        int mu = std::abs(mp - m);
        cplx sum(0, 0);
        if (tau == taup) {
            for (int p = std::abs(l - lp); p <= l + lp; ++p)
                sum += T.a[T.idx(lp, mp, l, m, p)] * z[p] * leg[(size_t)p * P + mu];
        } else {
            for (int p = std::abs(l - lp) + 1; p <= l + lp; ++p)
                sum += T.b[T.idx(lp, mp, l, m, p)] * z[p] * leg[(size_t)p * P + mu];
        }
        W[(size_t)nindex(lmax, tau, l, m) * nmax + nindex(lmax, taup, lp, mp)] =
            phase[(mp - m) + P - 1] * sum;
    }
}

extern "C" {

double oracle_wigner3j(int j1, int j2, int j3, int m1, int m2, int m3) { return wigner3j(j1, j2, j3, m1, m2, m3); }

void oracle_a5(int l, int m, int lp, int mp, int p, double* out2) {
    cplx v = a5(l, m, lp, mp, p); out2[0] = v.real(); out2[1] = v.imag();
}
void oracle_b5(int l, int m, int lp, int mp, int p, double* out2) {
    cplx v = b5(l, m, lp, mp, p); out2[0] = v.real(); out2[1] = v.imag();
}
double oracle_legendre_normalized(int l, int m, double x) { return legendre_normalized(l, m, x); }

void oracle_radial(int kind, int p, double x, double* out2) {
    cplx v = radial(kind, p, x); out2[0] = v.real(); out2[1] = v.imag();
}

// A_{nn'}(d) of (A.6)-(A.8) evaluated term by term, nothing cached.  kind: 3 = h^(1), 1 = j, 2 = y.
void oracle_translation_A(int tau, int l, int m, int taup, int lp, int mp, double k,
                          double dx, double dy, double dz, int kind, double* out2) {
    cplx v = translation_A(tau, l, m, taup, lp, mp, k, dx, dy, dz, kind);
    out2[0] = v.real(); out2[1] = v.imag();
}

// W block (eq. 7) for d = r_i - r_i'; W is nmax*nmax complex128, row-major [n][n'].
void oracle_coupling_block(int lmax, double k, double dx, double dy, double dz, int kind, double* W) {
    CoefTable T(lmax);
    coupling_block(T, k, dx, dy, dz, kind, reinterpret_cast<cplx*>(W));
}

// y^i_n = sum_{i' != i} sum_{n'} W^{ii'}_{nn'} b^{i'}_{n'}   (eq. 6 without a_in) for the listed receivers.
//   pos  [N][3] double, b [N][nmax] complex128, recv [n_recv] sphere indices, y [n_recv][nmax] complex128.
// Returns the number of OpenMP threads used.
int oracle_coupling_matvec(int N, int lmax, double k, const double* pos, const double* b_,
                           int n_recv, const int64_t* recv, double* y_, int kind) {
    const int nmax = 2 * lmax * (lmax + 2);
    const cplx* b = reinterpret_cast<const cplx*>(b_);
    cplx* y = reinterpret_cast<cplx*>(y_);
    CoefTable T(lmax);
    int nthreads = 1;
#pragma omp parallel
    {
#ifdef _OPENMP
#pragma omp single
        nthreads = omp_get_num_threads();
#endif
        std::vector<cplx> W((size_t)nmax * nmax);
#pragma omp for schedule(dynamic, 1)
        for (int r = 0; r < n_recv; ++r) {
            const int i = (int)recv[r];
            std::vector<cplx> acc(nmax, cplx(0, 0));
            for (int ip = 0; ip < N; ++ip) {
                if (ip == i) continue;                                   // sum over i' != i
                coupling_block(T, k, pos[3 * i] - pos[3 * ip], pos[3 * i + 1] - pos[3 * ip + 1],
                               pos[3 * i + 2] - pos[3 * ip + 2], kind, W.data());
                for (int n = 0; n < nmax; ++n) {
                    cplx s(0, 0);
                    for (int np = 0; np < nmax; ++np) s += W[(size_t)n * nmax + np] * b[(size_t)ip * nmax + np];
                    acc[n] += s;
                }
            }
            for (int n = 0; n < nmax; ++n) y[(size_t)r * nmax + n] = acc[n];
        }
    }
    return nthreads;
}

}  // extern "C"
