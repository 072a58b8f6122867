#!/usr/bin/env python3
"""Generator of the rotate / axial-translate / rotate pair body of the coupling kernel.

Writes ``generated/coupling_rot_lmax{L}.inc`` (L = 1..4): straight-line C++ device code, every constant a float
literal.  The paper mentions this factorisation as the O(lmax^3) alternative to its direct O(lmax^4) sum
(PAPER.md:185); BASELINE.json's north_star allows it "if it matches the oracle".

Formulation.  For the ordered pair (receiver i, emitter i'), d = r_i - r_i' with
spherical coordinates (d, theta, phi):

    W(d) = D^H  Wz(kd)  D,      D = blockdiag_{tau,l} D^l,   D^l_{m'm} = g(m') g(m) d^l_{m'm}(theta) e^{i m phi},

with d^l the Wigner small-d matrix, g(m) = (-1)^m for m < 0 and 1 otherwise (the gauge that goes with the
normalised Legendre functions WITHOUT Condon-Shortley phase), and Wz(kd) the coupling block for a
translation along +z, which is diagonal in m (only P_p^0(1) = sqrt((2p+1)/2) survives in (A.7)-(A.8)):

    Wz_{(tau l m),(tau' l' m)} = sum_p c_p h_p(kd) sqrt((2p+1)/2),  c_p = a5(l',m|l,m|p) or b5(l',m|l,m|p).

The kernel works in an orthonormal basis in which all of this is block diagonal with REAL rotation blocks:
    tau:  x_S = (x_1 + x_2)/sqrt2, x_A = (x_1 - x_2)/sqrt2        -> Wz = diag(A + B, A - B)
    m:    u+_m = (x_m + x_-m)/sqrt2, u-_m = (x_m - x_-m)/sqrt2, u_0 -> R = g d g splits into R+ ((l+1)^2) and R- (l^2)
(the pack / finalize kernels convert b and y; layout per tau block and l: [u_0, u+_1, u-_1, ..., u+_l, u-_l]).
Per pair:  (1) z-rotation  u~+ = cos(m phi) u+ + i sin(m phi) u-,  u~- = i sin(m phi) u+ + cos(m phi) u-;
           (2) u' = R+- u~;   (3) y'+ = A u'+ +- B u'-,  y'- = A u'- +- B u'+  (sign: tau block S / A);
           (4) v = R+-^T y';  (5) y+ += cos v+ - i sin v-,  y- += -i sin v+ + cos v-.

The rotation blocks are polynomials in cos(theta), sin(theta) obtained here symbolically with SymPy from the
closed form of d^l; a5/b5 come from gen_coupling_body.a5_b5 (exact SymPy Wigner-3j).  Nothing is shared with
oracle/.   Usage:  python gen_rotated_body.py [lmax ...]     (default 1 2 3 4)
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


def emit(lmax, outdir=None):
    H = lmax * (lmax + 2)
    P = 2 * lmax + 1
    out = []
    w = out.append
    coef = axial_tables(lmax)
    w(f"// AUTO-GENERATED by gen_rotated_body.py for lmax = {lmax} -- do not edit.")
    w("// Rotate / axial-translate / rotate pair body; see the generator's docstring for the formulation.")
    w("template <>")
    w(f"struct PairBodyRot<{lmax}> {{")
    w(f"  static constexpr int H = {H};")
    w(f"  static constexpr int P = {P};")
    w("  // hr/hi: h_p^(1)(kd); ct/st: cos/sin theta_d; cph/sph: cos/sin phi_d; bload(q): emitter coefficient q in the")
    w("  // orthonormal [tau S|A][l][u_0,u+_1,u-_1,...] basis; yacc(q, re, im): accumulate receiver coefficient q.")
    w("  template <class BLoad, class YAcc>")
    w("  CELES_DEVICE static void run(const float* hr, const float* hi, float ct, float st, float cph, float sph,")
    w("                               const BLoad& bload, YAcc& yacc) {")
    # phases
    w(f"    float cm[{lmax + 1}], sm[{lmax + 1}];")
    w("    cm[0] = 1.0f; sm[0] = 0.0f; cm[1] = cph; sm[1] = sph;")
    for m in range(2, lmax + 1):
        w(f"    cm[{m}] = fmaf(cm[{m - 1}], cph, -sm[{m - 1}] * sph); sm[{m}] = fmaf(cm[{m - 1}], sph, sm[{m - 1}] * cph);")
    # rotation blocks
    nrot = 0
    for l in range(1, lmax + 1):
        Rp, Rm = rotation_blocks(l)
        for name, blk in (("p", Rp), ("m", Rm)):
            for i, row in enumerate(blk):
                for j, (cf, spow) in enumerate(row):
                    var = f"R{name}{l}_{i}_{j}"
                    if len(cf) == 1:
                        expr = flit(cf[0])
                        if spow:
                            expr = f"{flit(cf[0])} * st"
                    else:
                        expr = flit(cf[0])
                        for a in cf[1:]:
                            expr = f"fmaf({expr}, ct, {flit(a)})"
                        if spow:
                            expr = f"({expr}) * st"
                    w(f"    const float {var} = {expr};")
                    nrot += 1
    # axial translation coefficients (shared by both tau blocks)
    for (l, lp, m), (A, B) in coef.items():
        for name, terms in (("A", A), ("B", B)):
            if not terms:
                continue
            p0, c0 = terms[0]
            var = f"{name}{l}{lp}{m}"
            er, ei = f"{flit(c0)} * hr[{p0}]", f"{flit(c0)} * hi[{p0}]"
            for (p, cc) in terms[1:]:
                er = f"fmaf({flit(cc)}, hr[{p}], {er})"
                ei = f"fmaf({flit(cc)}, hi[{p}], {ei})"
            if name == "A":
                w(f"    const float {var}r = {er}, {var}i = {ei};")
            else:
                # B = i * (beta_r + i beta_i) = -beta_i + i beta_r
                w(f"    const float {var}i = {er}, {var}t = {ei}; const float {var}r = -{var}t;")

    def mac(acc, kr, ki, xr, xi, first, sign=""):
        """acc (+)= sign (kr + i ki) (xr + i xi)"""
        if sign == "-":
            if first:
                w(f"      {acc}r = fmaf({ki}, {xi}, -({kr} * {xr})); {acc}i = -fmaf({kr}, {xi}, {ki} * {xr});")
            else:
                w(f"      {acc}r = fmaf(-{kr}, {xr}, {acc}r); {acc}r = fmaf({ki}, {xi}, {acc}r);")
                w(f"      {acc}i = fmaf(-{kr}, {xi}, {acc}i); {acc}i = fmaf(-{ki}, {xr}, {acc}i);")
        else:
            if first:
                w(f"      {acc}r = fmaf(-{ki}, {xi}, {kr} * {xr}); {acc}i = fmaf({kr}, {xi}, {ki} * {xr});")
            else:
                w(f"      {acc}r = fmaf({kr}, {xr}, {acc}r); {acc}r = fmaf(-{ki}, {xi}, {acc}r);")
                w(f"      {acc}i = fmaf({kr}, {xi}, {acc}i); {acc}i = fmaf({ki}, {xr}, {acc}i);")

    for ts in (0, 1):
        sg = "" if ts == 0 else "-"
        w(f"    {{ // tau block {'S = (1+2)/sqrt2' if ts == 0 else 'A = (1-2)/sqrt2'}")
        # (1)+(2): load, z-rotate, y-rotate
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            w(f"      const float2 b{l}_0 = bload({o});")
            w(f"      const float zp{l}_0r = b{l}_0.x, zp{l}_0i = b{l}_0.y;")
            for m in range(1, l + 1):
                w(f"      const float2 bp{l}_{m} = bload({o + 2 * m - 1}), bm{l}_{m} = bload({o + 2 * m});")
                w(f"      const float zp{l}_{m}r = fmaf(cm[{m}], bp{l}_{m}.x, -sm[{m}] * bm{l}_{m}.y), "
                  f"zp{l}_{m}i = fmaf(cm[{m}], bp{l}_{m}.y, sm[{m}] * bm{l}_{m}.x);")
                w(f"      const float zm{l}_{m}r = fmaf(cm[{m}], bm{l}_{m}.x, -sm[{m}] * bp{l}_{m}.y), "
                  f"zm{l}_{m}i = fmaf(cm[{m}], bm{l}_{m}.y, sm[{m}] * bp{l}_{m}.x);")
            for mt in range(0, l + 1):
                for part in ("r", "i"):
                    e = f"Rp{l}_{mt}_0 * zp{l}_0{part}"
                    for m in range(1, l + 1):
                        e = f"fmaf(Rp{l}_{mt}_{m}, zp{l}_{m}{part}, {e})"
                    w(f"      const float up{l}_{mt}{part} = {e};")
            for mt in range(1, l + 1):
                for part in ("r", "i"):
                    e = f"Rm{l}_{mt - 1}_0 * zm{l}_1{part}"
                    for m in range(2, l + 1):
                        e = f"fmaf(Rm{l}_{mt - 1}_{m - 1}, zm{l}_{m}{part}, {e})"
                    w(f"      const float um{l}_{mt}{part} = {e};")
        # (3) axial translation
        for l in range(1, lmax + 1):
            for mt in range(0, l + 1):
                w(f"      float yp{l}_{mt}r, yp{l}_{mt}i;" + (f" float ym{l}_{mt}r, ym{l}_{mt}i;" if mt else ""))
                first_p, first_m = True, True
                for lp in range(max(1, mt), lmax + 1):
                    A, B = coef[(l, lp, mt)]
                    if A:
                        mac(f"yp{l}_{mt}", f"A{l}{lp}{mt}r", f"A{l}{lp}{mt}i", f"up{lp}_{mt}r", f"up{lp}_{mt}i", first_p)
                        first_p = False
                        if mt:
                            mac(f"ym{l}_{mt}", f"A{l}{lp}{mt}r", f"A{l}{lp}{mt}i", f"um{lp}_{mt}r", f"um{lp}_{mt}i", first_m)
                            first_m = False
                    if B and mt:
                        mac(f"yp{l}_{mt}", f"B{l}{lp}{mt}r", f"B{l}{lp}{mt}i", f"um{lp}_{mt}r", f"um{lp}_{mt}i", first_p, sg)
                        first_p = False
                        mac(f"ym{l}_{mt}", f"B{l}{lp}{mt}r", f"B{l}{lp}{mt}i", f"up{lp}_{mt}r", f"up{lp}_{mt}i", first_m, sg)
                        first_m = False
                assert not first_p and (mt == 0 or not first_m)
        # (4)+(5): rotate back and accumulate
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            for m in range(0, l + 1):
                for part in ("r", "i"):
                    e = f"Rp{l}_0_{m} * yp{l}_0{part}"
                    for mt in range(1, l + 1):
                        e = f"fmaf(Rp{l}_{mt}_{m}, yp{l}_{mt}{part}, {e})"
                    w(f"      const float vp{l}_{m}{part} = {e};")
            for m in range(1, l + 1):
                for part in ("r", "i"):
                    e = f"Rm{l}_0_{m - 1} * ym{l}_1{part}"
                    for mt in range(2, l + 1):
                        e = f"fmaf(Rm{l}_{mt - 1}_{m - 1}, ym{l}_{mt}{part}, {e})"
                    w(f"      const float vm{l}_{m}{part} = {e};")
            w(f"      yacc({o}, vp{l}_0r, vp{l}_0i);")
            for m in range(1, l + 1):
                # y+ += c v+ - i s v-  ;  y- += -i s v+ + c v-
                w(f"      yacc({o + 2 * m - 1}, fmaf(cm[{m}], vp{l}_{m}r, sm[{m}] * vm{l}_{m}i), "
                  f"fmaf(cm[{m}], vp{l}_{m}i, -sm[{m}] * vm{l}_{m}r));")
                w(f"      yacc({o + 2 * m}, fmaf(cm[{m}], vm{l}_{m}r, sm[{m}] * vp{l}_{m}i), "
                  f"fmaf(cm[{m}], vm{l}_{m}i, -sm[{m}] * vp{l}_{m}r));")
        w("    }")
    w("  }")
    w("};")
    outdir = outdir or os.path.join(HERE, "generated")
    os.makedirs(outdir, exist_ok=True)
    path = os.path.join(outdir, f"coupling_rot_lmax{lmax}.inc")
    with open(path, "w") as f:
        f.write("\n".join(out) + "\n")
    print(f"lmax={lmax}: {nrot} rotation entries, {len(coef)} axial (l,l',m) entries -> {path}")


if __name__ == "__main__":
    for L in ([int(a) for a in sys.argv[1:]] or [1, 2, 3, 4]):
        emit(L)
