#!/usr/bin/env python3
"""Generator of the PACKED rotate / axial-translate / rotate pair body of the coupling kernel (sm_100a FFMA2).

Writes ``generated/coupling_pk_lmax{L}.inc`` (L = 1..4): straight-line C++ device code in which every complex
number is one ``float2`` (re, im) and every arithmetic step is a packed ``fma.rn.f32x2`` / ``mul.rn.f32x2`` /
``add.rn.f32x2`` (SASS FFMA2 / FMUL2 / FADD2, Blackwell only): a real coefficient times a complex value is ONE
instruction with the coefficient as a broadcast scalar operand, a complex times complex product is TWO (the
second one with the swapped-halves operand form and a (-,+) sign pattern).  Same FP32 work on the FMA pipe as the
scalar body of gen_rotated_body.py, about half the issue slots.

Formulation: that of gen_rotated_body.py (W(d) = D^H Wz(kd) D, PAPER.md:185 names the factorisation; Wz from
(A.7)-(A.8) with P_p^0(1) = sqrt((2p+1)/2)) with three changes:

  * the "minus" components are carried as w_m = i u-_m (pack / finalize kernels convert), which makes the
    z-rotation a REAL plane rotation of (u+_m, w_m):   u~+ = c u+ + s w,  w~ = c w - s u+   (c, s = cos, sin m phi);
    the axial step becomes  y'+ = A u'+ +- beta w',  y'w = A w' -+ beta u'+  (B = i beta, sign = tau block S / A),
    which for m >= 1 is diagonal on g+- = u'+ -+ i w' with eigenvalues A +- i s beta (half the complex products);
  * only the unique rotation entries are evaluated: R+-[j][i] = +- R+-[i][j] (d^l_{m'm} = (-1)^{m-m'} d^l_{mm'}),
    detected numerically here, as polynomials in cos^2(theta) times cos / sin factors;
  * the axial coefficients obey A_{l'l m} = +- A_{ll'm}, beta_{l'l m} = +- beta_{ll'm} (detected numerically):
    only l <= l' is evaluated, as packed sums  sum_p c_p (Re h_p, Im h_p).

Nothing is shared with oracle/.   Usage:  python gen_packed_body.py [lmax ...]     (default 1 2 3 4)
"""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from gen_coupling_body import flit  # noqa: E402
from gen_rotated_body import axial_tables, rotation_blocks  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
TOL = 1e-12


def poly_key(cf, spow):
    """canonical form of a rotation entry: (coefficients high->low with leading zeros removed, s power)"""
    c = list(cf)
    while len(c) > 1 and abs(c[0]) < TOL:
        c.pop(0)
    return tuple(c), spow


def related(e1, e2):
    """+1 / -1 if entry e1 == +- e2, else 0"""
    (c1, s1), (c2, s2) = e1, e2
    if s1 != s2 or len(c1) != len(c2):
        return 0
    for sign in (1, -1):
        if all(abs(a - sign * b) <= TOL * max(1.0, abs(a)) for a, b in zip(c1, c2)):
            return sign
    return 0


class Entries:
    """Unique rotation entries -> C expressions.  ref(name) returns (sign, expr) with expr a float variable,
    'ct', 'st', or None for the constants +-1 (sign carries it) / zero (sign 0)."""

    def __init__(self, w):
        self.w = w
        self.defs = []          # (canonical entry, variable)
        self.n_ops = 0

    def ref(self, cf, spow, hint):
        key = poly_key(cf, spow)
        c, sp = key
        if all(abs(a) < TOL for a in c):
            return 0, None
        if sp == 0 and len(c) == 1:                       # constant
            if abs(abs(c[0]) - 1.0) < TOL:
                return (1 if c[0] > 0 else -1), None
        if sp == 0 and len(c) == 2 and abs(c[1]) < TOL and abs(abs(c[0]) - 1.0) < TOL:
            return (1 if c[0] > 0 else -1), "ct"          # +- cos(theta)
        if sp == 1 and len(c) == 1 and abs(abs(c[0]) - 1.0) < TOL:
            return (1 if c[0] > 0 else -1), "st"          # +- sin(theta)
        if sp == 1 and len(c) == 2 and abs(c[1]) < TOL and abs(abs(c[0]) - 1.0) < TOL:
            return (1 if c[0] > 0 else -1), "cst"         # +- cos(theta) sin(theta)
        for k, var in self.defs:
            s = related(key, k)
            if s:
                return s, var
        var = hint
        self.defs.append((key, var))
        self.w(f"    const float {var} = {self.expr(c, sp)};")
        return 1, var

    def expr(self, c, sp):
        """polynomial of one parity in ct (checked) evaluated by Horner in c2 = ct*ct, times ct and/or st"""
        deg = len(c) - 1
        par = deg % 2
        for k, a in enumerate(c):
            if (deg - k) % 2 != par:
                assert abs(a) < TOL, "rotation entry of mixed parity in cos(theta)"
        terms = [a for k, a in enumerate(c) if (deg - k) % 2 == par]      # in powers of c2, high -> low
        e = flit(terms[0])
        for a in terms[1:]:
            e = f"fmaf({e}, c2, {flit(a)})"
            self.n_ops += 1
        fac = {(0, 0): None, (1, 0): "ct", (0, 1): "st", (1, 1): "cst"}[(par, sp)]
        if fac:
            if len(terms) == 1:
                e = f"{flit(terms[0])} * {fac}"
            else:
                e = f"({e}) * {fac}"
            self.n_ops += 1
        return e


def bcast(sign, var):
    """broadcast operand (both halves) of a signed scalar"""
    return f"bc2({'-' if sign < 0 else ''}{var})"


def emit(lmax, outdir=None):
    H = lmax * (lmax + 2)
    P = 2 * lmax + 1
    out = []
    w = out.append
    coef = axial_tables(lmax)
    w(f"// AUTO-GENERATED by gen_packed_body.py for lmax = {lmax} -- do not edit.")
    w("// Packed (FFMA2) rotate / axial-translate / rotate pair body; see the generator's docstring.")
    w("template <>")
    w(f"struct PairBodyPk<{lmax}> {{")
    w(f"  static constexpr int H = {H};")
    w(f"  static constexpr int P = {P};")
    w("  // h[p] = (Re, Im) h_p^(1)(kd); ct/st: cos/sin theta_d; cph/sph: cos/sin phi_d; bload(q): emitter coefficient q")
    w("  // (re, im) in the [tau S|A][l][u_0,u+_1,w_1,...] basis (w = i u-); yacc.get/put(q): receiver accumulator q.")
    w("  template <class BLoad, class YAcc>")
    w("  CELES_DEVICE static void run(const float2* h, float ct, float st, float cph, float sph,")
    w("                               const BLoad& bload, YAcc& yacc) {")
    w(f"    float cm[{lmax + 1}], sm[{lmax + 1}];")
    w("    cm[0] = 1.0f; sm[0] = 0.0f; cm[1] = cph; sm[1] = sph;")
    for m in range(2, lmax + 1):
        w(f"    cm[{m}] = fmaf(cm[{m - 1}], cph, -sm[{m - 1}] * sph); sm[{m}] = fmaf(cm[{m - 1}], sph, sm[{m - 1}] * cph);")
    w("    const float c2 = ct * ct, cst = ct * st; (void)c2; (void)cst;")
    # ---- rotation entries (unique ones only)
    ent = Entries(w)
    R = {}
    for l in range(1, lmax + 1):
        Rp, Rm = rotation_blocks(l)
        for name, blk in (("p", Rp), ("m", Rm)):
            for i, row in enumerate(blk):
                for j, (cf, spow) in enumerate(row):
                    R[(name, l, i, j)] = ent.ref(cf, spow, f"R{name}{l}_{i}_{j}")
    # ---- axial coefficients, unique (l <= l') ones, packed (re, im)
    ax = {}
    n_ax_ops = 0

    def same(u, v):
        if len(u) != len(v) or any(pu != pv for (pu, _), (pv, _) in zip(u, v)):
            return 0
        for sign in (1, -1):
            if all(abs(cu - sign * cv) <= 1e-12 * max(1.0, abs(cu)) for (_, cu), (_, cv) in zip(u, v)):
                return sign
        return 0

    for (l, lp, m), (A, B) in coef.items():
        for name, terms in (("A", A), ("B", B)):
            if not terms:
                ax[(name, l, lp, m)] = (0, None)
                continue
            if l > lp:
                s = same(terms, coef[(lp, l, m)][0 if name == "A" else 1])
                assert s != 0, "axial coefficients are not (anti)symmetric in (l, l')"
                ax[(name, l, lp, m)] = (s, f"{name}{lp}{l}{m}")
                continue
            var = f"{name}{l}{lp}{m}"
            if m >= 1:
                terms = [(p, 0.5 * cc) for (p, cc) in terms]        # eigenvalues (A +- i beta) / 2 below
            p0, c0 = terms[0]
            if abs(abs(c0) - 1.0) < TOL:
                e = f"h[{p0}]" if c0 > 0 else f"neg2(h[{p0}])"
                n_ax_ops -= 1
            else:
                e = f"mul2(bc2({flit(c0)}), h[{p0}])"
            for (p, cc) in terms[1:]:
                e = f"fma2(bc2({flit(cc)}), h[{p}], {e})"
            n_ax_ops += len(terms)
            w(f"    const float2 {var} = {e};")
            ax[(name, l, lp, m)] = (1, var)
        if m >= 1 and l <= lp:
            # m >= 1: the (u+, w) 2x2 block [[A, s beta], [-s beta, A]] has eigenvectors (1, +-i), eigenvalues A +- i s beta
            assert A and B
            w(f"    const float2 E{l}{lp}{m}a = add2(A{l}{lp}{m}, make_float2(-B{l}{lp}{m}.y, B{l}{lp}{m}.x));")
            w(f"    const float2 E{l}{lp}{m}b = add2(A{l}{lp}{m}, make_float2(B{l}{lp}{m}.y, -B{l}{lp}{m}.x));")

    def cmac(acc, sign, kvar, x, first):
        """(P, Q) (+)= sign * (k.x, k.y) * x: the complex product k x = P + i Q is kept as two packed sums with a
        broadcast scalar coefficient each (no swapped / sign-patterned operands); combined once per output."""
        sg = "-" if sign < 0 else ""
        if first:
            w(f"      float2 {acc}P = mul2(bc2({sg}{kvar}.x), {x}), {acc}Q = mul2(bc2({sg}{kvar}.y), {x});")
        else:
            w(f"      {acc}P = fma2(bc2({sg}{kvar}.x), {x}, {acc}P); {acc}Q = fma2(bc2({sg}{kvar}.y), {x}, {acc}Q);")

    def rsum(terms):
        """sum of (sign, var, x): real coefficient times packed complex; var None means the constant 1"""
        plain = [(s, x) for (s, v, x) in terms if v is None and s != 0]
        mult = [(s, v, x) for (s, v, x) in terms if v is not None and s != 0]
        e = None
        for (s, v, x) in mult:
            e = f"mul2({bcast(s, v)}, {x})" if e is None else f"fma2({bcast(s, v)}, {x}, {e})"
        for (s, x) in plain:
            if e is None:
                e = x if s > 0 else f"neg2({x})"
            else:
                e = f"add2({e}, {x})" if s > 0 else f"sub2({e}, {x})"
        assert e is not None
        return e

    for ts in (0, 1):
        tsign = 1 if ts == 0 else -1
        w(f"    {{ // tau block {'S = (1+2)/sqrt2' if ts == 0 else 'A = (1-2)/sqrt2'}")
        # (1) load + z-rotation (real plane rotation of (u+_m, w_m)), (2) y-rotation
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            w(f"      const float2 zp{l}_0 = bload({o});")
            for m in range(1, l + 1):
                w(f"      const float2 bp{l}_{m} = bload({o + 2 * m - 1}), bw{l}_{m} = bload({o + 2 * m});")
                w(f"      const float2 zp{l}_{m} = fma2(bc2(cm[{m}]), bp{l}_{m}, mul2(bc2(sm[{m}]), bw{l}_{m}));")
                w(f"      const float2 zw{l}_{m} = fma2(bc2(cm[{m}]), bw{l}_{m}, mul2(bc2(-sm[{m}]), bp{l}_{m}));")
            for mt in range(0, l + 1):
                terms = [(*R[("p", l, mt, m)], f"zp{l}_{m}") for m in range(0, l + 1)]
                w(f"      const float2 up{l}_{mt} = {rsum(terms)};")
            for mt in range(1, l + 1):
                terms = [(*R[("m", l, mt - 1, m - 1)], f"zw{l}_{m}") for m in range(1, l + 1)]
                w(f"      const float2 uw{l}_{mt} = {rsum(terms)};")
        # (3) axial translation.  m = 0: y'+ = A u'+.  m >= 1: y'+ = A u'+ +- beta w', y'w = A w' -+ beta u'+ is
        # diagonal on g+- = u'+ -+ i w':  y'+ = L+ g+ + L- g-,  y'w = i (L+ g+ - L- g-),  L+- = (A +- i s beta) / 2
        for mt in range(1, lmax + 1):
            for lp in range(mt, lmax + 1):
                w(f"      const float2 gp{lp}_{mt} = add2(up{lp}_{mt}, make_float2(uw{lp}_{mt}.y, -uw{lp}_{mt}.x));")
                w(f"      const float2 gm{lp}_{mt} = add2(up{lp}_{mt}, make_float2(-uw{lp}_{mt}.y, uw{lp}_{mt}.x));")
        for l in range(1, lmax + 1):
            first = True
            for lp in range(1, lmax + 1):
                sa, va = ax[("A", l, lp, 0)]
                if sa:
                    cmac(f"yp{l}_0", sa, va, f"up{lp}_0", first)
                    first = False
            assert not first
            w(f"      const float2 yp{l}_0 = add2(yp{l}_0P, make_float2(-yp{l}_0Q.y, yp{l}_0Q.x));")
            for mt in range(1, l + 1):
                first = True
                for lp in range(mt, lmax + 1):
                    sa, va = ax[("A", l, lp, mt)]
                    sb, vb = ax[("B", l, lp, mt)]
                    assert sa and sb and va[1:] == vb[1:]
                    base = "E" + va[1:]
                    plus, minus = ("a", "b") if sa * sb * tsign > 0 else ("b", "a")
                    cmac(f"zp{l}_{mt}", sa, base + plus, f"gp{lp}_{mt}", first)
                    cmac(f"zm{l}_{mt}", sa, base + minus, f"gm{lp}_{mt}", first)
                    first = False
                w(f"      const float2 zp{l}_{mt}c = add2(zp{l}_{mt}P, make_float2(-zp{l}_{mt}Q.y, zp{l}_{mt}Q.x));")
                w(f"      const float2 zm{l}_{mt}c = add2(zm{l}_{mt}P, make_float2(-zm{l}_{mt}Q.y, zm{l}_{mt}Q.x));")
                w(f"      const float2 yp{l}_{mt} = add2(zp{l}_{mt}c, zm{l}_{mt}c);")
                w(f"      const float2 yw{l}_{mt} = add2(make_float2(-zp{l}_{mt}c.y, zp{l}_{mt}c.x), make_float2(zm{l}_{mt}c.y, -zm{l}_{mt}c.x));")
        # (4) rotate back (transposes), (5) z-rotate back and accumulate
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            for m in range(0, l + 1):
                terms = [(*R[("p", l, mt, m)], f"yp{l}_{mt}") for mt in range(0, l + 1)]
                if m == 0:
                    w(f"      yacc.put({o}, add2(yacc.get({o}), {rsum(terms)}));")
                else:
                    w(f"      const float2 vp{l}_{m} = {rsum(terms)};")
            for m in range(1, l + 1):
                terms = [(*R[("m", l, mt - 1, m - 1)], f"yw{l}_{mt}") for mt in range(1, l + 1)]
                w(f"      const float2 vw{l}_{m} = {rsum(terms)};")
            for m in range(1, l + 1):
                # y+ += c v+ - s vw ;  yw += s v+ + c vw
                qp, qw = o + 2 * m - 1, o + 2 * m
                w(f"      yacc.put({qp}, fma2(bc2(-sm[{m}]), vw{l}_{m}, fma2(bc2(cm[{m}]), vp{l}_{m}, yacc.get({qp}))));")
                w(f"      yacc.put({qw}, fma2(bc2(cm[{m}]), vw{l}_{m}, fma2(bc2(sm[{m}]), vp{l}_{m}, yacc.get({qw}))));")
        w("    }")
    w("  }")
    w("};")
    outdir = outdir or os.path.join(HERE, "generated")
    os.makedirs(outdir, exist_ok=True)
    path = os.path.join(outdir, f"coupling_pk_lmax{lmax}.inc")
    with open(path, "w") as f:
        f.write("\n".join(out) + "\n")
    print(f"lmax={lmax}: {len(ent.defs)} unique rotation entries ({ent.n_ops} scalar ops), "
          f"{n_ax_ops} packed axial-coefficient terms -> {path}")


if __name__ == "__main__":
    for L in ([int(a) for a in sys.argv[1:]] or [1, 2, 3, 4]):
        emit(L)
