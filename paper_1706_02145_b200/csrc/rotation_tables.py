#!/usr/bin/env python3
"""Symbolic tables of the rotate / axial-translate / rotate factorisation of the coupling block (used by
gen_packed_body.py).  The paper mentions this factorisation as the O(lmax^3) alternative to its direct O(lmax^4) sum
(PAPER.md:185); BASELINE.json's north_star allows it "if it matches the oracle".

Formulation.  For the ordered pair (receiver i, emitter i'), d = r_i - r_i' with
spherical coordinates (d, theta, phi):

    W(d) = D^H  Wz(kd)  D,      D = blockdiag_{tau,l} D^l,   D^l_{m'm} = g(m') g(m) d^l_{m'm}(theta) e^{i m phi},

with d^l the Wigner small-d matrix, g(m) = (-1)^m for m < 0 and 1 otherwise (the gauge that goes with the
normalised Legendre functions WITHOUT Condon-Shortley phase), and Wz(kd) the coupling block for a
translation along +z, which is diagonal in m (only P_p^0(1) = sqrt((2p+1)/2) survives in (A.7)-(A.8)):

    Wz_{(tau l m),(tau' l' m)} = sum_p c_p h_p(kd) sqrt((2p+1)/2),  c_p = a5(l',m|l,m|p) or b5(l',m|l,m|p).

In the orthonormal basis
    tau:  x_S = (x_1 + x_2)/sqrt2, x_A = (x_1 - x_2)/sqrt2        -> Wz = diag(A + B, A - B)
    m:    u+_m = (x_m + x_-m)/sqrt2, u-_m = (x_m - x_-m)/sqrt2, u_0 -> R = g d g splits into R+ ((l+1)^2) and R- (l^2)
all of this is block diagonal with REAL rotation blocks.  ``rotation_blocks(l)`` returns R+ and R- as polynomials in
cos(theta) times sin(theta)^(0|1), obtained symbolically with SymPy from the closed form of d^l; ``axial_tables(lmax)``
the real coefficients of the sums over p of Wz, from gen_coupling_body.a5_b5 (exact SymPy Wigner-3j).
Nothing is shared with oracle/.
"""
import math
import os
import sys

import sympy as sp

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from gen_coupling_body import a5_b5, flit  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
C, S = sp.symbols("c s", real=True)


def half_angle_monomial(a, b):
    """cos(theta/2)^a sin(theta/2)^b (a + b even) as a polynomial in c = cos(theta) times s^(0|1)."""
    q = min(a, b)
    expr = (S / 2) ** q
    if a > b:
        expr *= ((1 + C) / 2) ** ((a - b) // 2)
    elif b > a:
        expr *= ((1 - C) / 2) ** ((b - a) // 2)
    return expr


def small_d(l):
    """Wigner small-d matrix d^l_{m'm}(theta), symbolic in (c, s); dict keyed (m', m)."""
    f = sp.factorial
    out = {}
    for mp in range(-l, l + 1):
        for m in range(-l, l + 1):
            tot = 0
            for k in range(max(0, m - mp), min(l + m, l - mp) + 1):
                num = (-1) ** (k - m + mp) * sp.sqrt(f(l + m) * f(l - m) * f(l + mp) * f(l - mp))
                den = f(l + m - k) * f(k) * f(l - k - mp) * f(k - m + mp)
                tot += num / den * half_angle_monomial(2 * l - 2 * k + m - mp, 2 * k - m + mp)
            out[(mp, m)] = tot
    return out


def reduce_cs(expr):
    """expand and reduce s^2 -> 1 - c^2; returns (poly_in_c coefficients high->low, s_power in {0,1})."""
    e = sp.expand(expr)
    p = sp.Poly(e, S)
    even, odd = 0, 0
    for (k,), coef in p.terms():
        term = coef * (1 - C**2) ** (k // 2)
        if k % 2:
            odd += term
        else:
            even += term
    even, odd = sp.expand(even), sp.expand(odd)
    assert even == 0 or odd == 0, "mixed parity in a rotation entry"
    if odd != 0:
        return [float(x) for x in sp.Poly(odd, C).all_coeffs()], 1
    if even == 0:
        return [0.0], 0
    return [float(x) for x in sp.Poly(even, C).all_coeffs()], 0


def gauge(m):
    return -1 if (m < 0 and m % 2) else 1


def rotation_blocks(l):
    """R+ [(l+1) x (l+1)], R- [l x l] of R = g d g in the orthonormal (u_0, u+_m | u-_m) basis, entries as
    (coeffs, s_power)."""
    d = small_d(l)
    R = {(mp, m): gauge(mp) * gauge(m) * d[(mp, m)] for mp in range(-l, l + 1) for m in range(-l, l + 1)}
    r2 = sp.sqrt(2)
    Rp = [[None] * (l + 1) for _ in range(l + 1)]
    Rm = [[None] * l for _ in range(l)]
    Rp[0][0] = reduce_cs(R[(0, 0)])
    for m in range(1, l + 1):
        Rp[0][m] = reduce_cs(r2 * R[(0, m)])
        Rp[m][0] = reduce_cs(r2 * R[(m, 0)])
        for mp in range(1, l + 1):
            Rp[mp][m] = reduce_cs(R[(mp, m)] + R[(mp, -m)])
            Rm[mp - 1][m - 1] = reduce_cs(R[(mp, m)] - R[(mp, -m)])
    # sanity: R commutes with the flip m -> -m (so the +/- blocks decouple)
    for mp in range(-l, l + 1):
        for m in range(-l, l + 1):
            assert sp.simplify(sp.expand(R[(mp, m)] - R[(-mp, -m)]).subs(S**2, 1 - C**2)) == 0
    return Rp, Rm


def axial_tables(lmax):
    """coef[(l, lp, m)] = (A terms [(p, a5 * sqrt((2p+1)/2))], B terms [(p, b5'' * sqrt((2p+1)/2))]),
    m >= 0, for Wz_{(l m),(l' m)} (argument swap of eq. 7)."""
    coef = {}
    for l in range(1, lmax + 1):
        for lp in range(1, lmax + 1):
            for m in range(0, min(l, lp) + 1):
                A, B = [], []
                for p in range(abs(l - lp), l + lp + 1):
                    a, b = a5_b5(lp, m, l, m, p)
                    assert abs(a.imag) < 1e-20 and abs(b.real) < 1e-20
                    f = math.sqrt((2 * p + 1) / 2.0)
                    if abs(a.real) > 1e-14:
                        A.append((p, a.real * f))
                    if abs(b.imag) > 1e-14:
                        B.append((p, b.imag * f))
                # the -m entry has the same a5 and the opposite b5 (checked, not assumed)
                if m > 0:
                    for p in range(abs(l - lp), l + lp + 1):
                        a, b = a5_b5(lp, m, l, m, p)
                        am, bm = a5_b5(lp, -m, l, -m, p)
                        assert abs(a - am) < 1e-13 and abs(b + bm) < 1e-13
                else:
                    assert not B
                coef[(l, lp, m)] = (A, B)
    return coef
