// translation_table.h -- host-side evaluation of the a5 / b5 translation coefficients (PAPER.md:258-267,
// (A.9)-(A.11)) at run time, as celes_setup's "efficiency ... not critical" table step.
//
// Independent of oracle/ (which has its own Racah code): here the Wigner-3j symbol with zero projections uses
// its closed form and the general symbol is obtained from Clebsch-Gordan-style binomial sums in exact
// integer-valued doubles.  The compiled kernels carry the same numbers as float immediates (written by
// gen_coupling_body.py from SymPy); tests/test_host_logic.py checks all three against each other.
#pragma once
#include <cmath>
#include <cstdlib>
#include <vector>

namespace celes {

inline double fact(int n) {
    static const std::vector<double> tab = [] {
        std::vector<double> t(64, 1.0);
        for (int i = 1; i < 64; ++i) t[i] = t[i - 1] * i;
        return t;
    }();
    return tab[n];
}

// ( j1 j2 j3 ; 0 0 0 ) closed form: zero for odd J = j1+j2+j3, else
// (-1)^g sqrt( (J-2j1)! (J-2j2)! (J-2j3)! / (J+1)! ) g! / ((g-j1)! (g-j2)! (g-j3)!),  g = J/2
inline double threej_000(int j1, int j2, int j3) {
    const int J = j1 + j2 + j3;
    if (J & 1) return 0.0;
    if (j3 > j1 + j2 || j3 < std::abs(j1 - j2)) return 0.0;
    const int g = J / 2;
    const double tri = fact(J - 2 * j1) * fact(J - 2 * j2) * fact(J - 2 * j3) / fact(J + 1);
    const double v = std::sqrt(tri) * fact(g) / (fact(g - j1) * fact(g - j2) * fact(g - j3));
    return (g & 1) ? -v : v;
}

// general ( j1 j2 j3 ; m1 m2 m3 ), sum over the admissible range of the Racah index only
inline double threej(int j1, int j2, int j3, int m1, int m2, int m3) {
    if (m1 + m2 + m3 != 0) return 0.0;
    if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m3) > j3) return 0.0;
    if (j3 > j1 + j2 || j3 < std::abs(j1 - j2)) return 0.0;
    const int tmin = std::max(0, std::max(j2 - j3 - m1, j1 - j3 + m2));
    const int tmax = std::min(j1 + j2 - j3, std::min(j1 - m1, j2 + m2));
    double s = 0.0;
    for (int t = tmin; t <= tmax; ++t) {
        const double den = fact(t) * fact(j3 - j2 + t + m1) * fact(j3 - j1 + t - m2) * fact(j1 + j2 - j3 - t) *
                           fact(j1 - t - m1) * fact(j2 - t + m2);
        s += ((t & 1) ? -1.0 : 1.0) / den;
    }
    const double tri = fact(j1 + j2 - j3) * fact(j1 - j2 + j3) * fact(-j1 + j2 + j3) / fact(j1 + j2 + j3 + 1);
    const double pre = std::sqrt(tri * fact(j1 + m1) * fact(j1 - m1) * fact(j2 + m2) * fact(j2 - m2) *
                                 fact(j3 + m3) * fact(j3 - m3));
    const int ph = std::abs(j1 - j2 - m3);
    return ((ph & 1) ? -1.0 : 1.0) * pre * s;
}

// real and imaginary unit powers: i^k = (re, im)
inline void ipow(int k, double* re, double* im) {
    static const double R[4] = {1, 0, -1, 0}, I[4] = {0, 1, 0, -1};
    const int r = ((k % 4) + 4) % 4;
    *re = R[r]; *im = I[r];
}

// Fills a5_re / b5_im for W_{(l m),(l' m')} = A_{(l' m'),(l m)}: index ((r*H)+c)*P + p, r = receiver (l,m),
// c = emitter (l',m').  a5 is real and b5 imaginary for every admissible argument; returns false if that
// ever fails numerically (it would mean the formulas were mistyped).
inline bool build_translation_table(int lmax, std::vector<double>& a5_re, std::vector<double>& b5_im) {
    const int H = lmax * (lmax + 2), P = 2 * lmax + 1;
    a5_re.assign((size_t)H * H * P, 0.0);
    b5_im.assign((size_t)H * H * P, 0.0);
    bool ok = true;
    for (int l = 1; l <= lmax; ++l) for (int m = -l; m <= l; ++m)            // receiver (second index of A)
    for (int lp = 1; lp <= lmax; ++lp) for (int mp = -lp; mp <= lp; ++mp) {  // emitter (first index of A)
        const int r = (l - 1) * (l + 1) + (m + l), c = (lp - 1) * (lp + 1) + (mp + lp);
        // A_{n'n}: in (A.7)-(A.11) the roles are (l,m) <- emitter (lp,mp), (l',m') <- receiver (l,m)
        const int L1 = lp, M1 = mp, L2 = l, M2 = m;
        for (int p = std::abs(L1 - L2); p <= L1 + L2; ++p) {
            double pr, pi;
            ipow(std::abs(M1 - M2) - std::abs(M1) - std::abs(M2) + L2 - L1 + p, &pr, &pi);
            const double sgn = ((M1 - M2) & 1) ? -1.0 : 1.0;
            const double common = std::sqrt((2.0 * L1 + 1) * (2.0 * L2 + 1) / (2.0 * L1 * (L1 + 1) * L2 * (L2 + 1)));
            const double w = threej(L1, L2, p, M1, -M2, M2 - M1);
            const double a = sgn * (L1 * (L1 + 1) + L2 * (L2 + 1) - p * (p + 1)) * std::sqrt(2.0 * p + 1) * common * w *
                             threej_000(L1, L2, p);
            double b = 0.0;
            if (p >= 1) {
                const double rad = (double)(L1 + L2 + 1 + p) * (L1 + L2 + 1 - p) * (p + L1 - L2) * (p - L1 + L2) * (2.0 * p + 1);
                if (rad > 0) b = sgn * std::sqrt(rad) * common * w * threej_000(L1, L2, p - 1);
            }
            const size_t idx = ((size_t)r * H + c) * P + p;
            a5_re[idx] = pr * a;
            b5_im[idx] = pi * b;
            if (std::fabs(pi * a) > 1e-12 || std::fabs(pr * b) > 1e-12) ok = false;
        }
    }
    return ok;
}

}  // namespace celes
