#!/usr/bin/env python3
"""Generator of the PACKED rotate / axial-translate / rotate pair body of the coupling kernel (sm_100a FFMA2).

Writes ``generated/coupling_pk_lmax{L}.inc`` (L = 1..5): straight-line C++ device code in which every complex
number is one ``float2`` (re, im) and every arithmetic step is a packed ``fma.rn.f32x2`` / ``mul.rn.f32x2``
(SASS FFMA2 / FMUL2, Blackwell only).  A real coefficient times a complex value is ONE instruction with the
coefficient as a broadcast scalar operand; a complex times complex multiply-add is TWO (``cfma2``): FFMA2 takes its
vector operands with swapped halves (``.LO_HI``) and the addend with a (-,+) / (+,-) sign pattern (``.NP``), so
c + k x = k.x x + [k.y x.swapped + c.NP].NP needs no shuffles and no separate addition.  Multiplications by +-i
(``imul2`` / ``nimul2``) are such operand forms too and cost nothing.

Formulation: rotation_tables.py (W(d) = D^H Wz(kd) D, PAPER.md:185 names the factorisation; Wz from (A.7)-(A.8) with
P_p^0(1) = sqrt((2p+1)/2)), arranged so that nearly every packed instruction is an FMA:

  * the "minus" components are carried as w_m = i u-_m (pack / finalize kernels convert), which makes the
    z-rotation a REAL plane rotation of (u+_m, w_m):   u~+ = c u+ + s w,  w~ = c w - s u+   (c, s = cos, sin m phi);
  * only the unique rotation entries are evaluated: R+-[j][i] = +- R+-[i][j] (d^l_{m'm} = (-1)^{m-m'} d^l_{mm'}),
    detected numerically here, as polynomials in cos^2(theta) times cos / sin factors;
  * for m >= 1 the axial step  y'+ = A u'+ +- beta w',  y'w = A w' -+ beta u'+  (B = i beta, sign = tau block S / A)
    is diagonal on g+- = u'+ -+ i w' with eigenvalues E+- = (A +- i beta) / 2.  g+ is the y-rotation chain of u'+
    SEEDED with -i w' (no addition), g- = g+ + 2 i w' (one FMA);  z+ = sum E g+,  y'+ = z+ + sum E' g- (the second
    chain seeded with the first),  y'w = i (2 z+ - y'+) (one FMA);
  * the axial coefficients obey A_{l'l m} = +- A_{ll'm}, beta_{l'l m} = +- beta_{ll'm} (detected numerically):
    only l <= l' is evaluated, as packed sums  A = sum_p c_p h_p,  E+ = A + sum_p c'_p (i h_p),  E- = 2 A - E+;
  * every chain that ends in an accumulator starts from it.

``python gen_packed_body.py --table`` prints the per-phase operation counts (profiles/r02_phase_table.md).
Nothing is shared with oracle/.   Usage:  python gen_packed_body.py [lmax ...]     (default 1 2 3 4 5)
"""
import os
import re
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from gen_coupling_body import flit  # noqa: E402
from rotation_tables import axial_tables, rotation_blocks  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
TOL = 1e-12
INTERLEAVE = os.environ.get('CELES_GEN_INTERLEAVE', '0') == '1'
_TAUVAR = re.compile(r'\b(zp|bp|bw|zw|up|uw|gp|gm|yp|zq|yw|vp|vw)(\d+_\d+)\b')


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


PHASES = ["phases e^{i m phi}", "rotation entries", "axial coefficients", "z-rotation in", "y-rotation in + g+-",
          "axial apply + recombination", "y-rotation back", "z-rotation back + accumulate"]
_OPS = {"fma2": re.compile(r"\bfma2\("), "mul2": re.compile(r"\bmul2\("), "add2": re.compile(r"\b(?:add2|sub2)\("),
        "cfma2": re.compile(r"\bcfma2\("), "cmul2": re.compile(r"\bcmul2\("), "fmaf": re.compile(r"\bfmaf\("),
        "smul": re.compile(r"(?<![\w.)])[\w.\[\]]+f? \* [\w.\[\]]+|\) \* \w+")}


def count_ops(line):
    """(packed FMA, packed MUL, packed ADD, scalar ops) of one emitted source line"""
    n = {k: len(r.findall(line)) for k, r in _OPS.items()}
    return (n["fma2"] + 2 * n["cfma2"] + n["cmul2"], n["mul2"] + n["cmul2"], n["add2"], n["fmaf"] + n["smul"])


def emit(lmax, outdir=None, table=None, interleave=INTERLEAVE):
    H = lmax * (lmax + 2)
    P = 2 * lmax + 1
    out = []
    counts = {ph: [0, 0, 0, 0] for ph in PHASES}

    def w(line, phase=None):
        out.append(line)
        if phase is not None:
            for k, v in enumerate(count_ops(line)):
                counts[phase][k] += v

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
        w(f"    cm[{m}] = fmaf(cm[{m - 1}], cph, -sm[{m - 1}] * sph); sm[{m}] = fmaf(cm[{m - 1}], sph, sm[{m - 1}] * cph);",
          PHASES[0])
    w("    const float c2 = ct * ct, cst = ct * st; (void)c2; (void)cst;", PHASES[1])
    # ---- rotation entries (unique ones only)
    ent = Entries(lambda line: w(line, PHASES[1]))
    R = {}
    for l in range(1, lmax + 1):
        Rp, Rm = rotation_blocks(l)
        for name, blk in (("p", Rp), ("m", Rm)):
            for i, row in enumerate(blk):
                for j, (cf, spow) in enumerate(row):
                    R[(name, l, i, j)] = ent.ref(cf, spow, f"R{name}{l}_{i}_{j}")
    # ---- axial coefficients, unique (l <= l') ones, packed (re, im)
    ax = {}

    def same(u, v):
        if len(u) != len(v) or any(pu != pv for (pu, _), (pv, _) in zip(u, v)):
            return 0
        for sign in (1, -1):
            if all(abs(cu - sign * cv) <= 1e-12 * max(1.0, abs(cu)) for (_, cu), (_, cv) in zip(u, v)):
                return sign
        return 0

    def hsum(terms, seed=None, times_i=False):
        """seed + sum_p c_p h_p (times_i: c_p (i h_p)), one packed instruction per term"""
        e = seed
        for (p, cc) in terms:
            x = f"imul2(h[{p}])" if times_i else f"h[{p}]"
            if e is None:
                if abs(cc - 1.0) < TOL and not times_i:
                    e = x
                else:
                    e = f"mul2(bc2({flit(cc)}), {x})"
            else:
                e = f"fma2(bc2({flit(cc)}), {x}, {e})"
        return e

    for (l, lp, m), (A, B) in coef.items():
        if l > lp:
            for name, terms in (("A", A), ("B", B)):
                if not terms:
                    ax[(name, l, lp, m)] = (0, None)
                    continue
                s = same(terms, coef[(lp, l, m)][0 if name == "A" else 1])
                assert s != 0, "axial coefficients are not (anti)symmetric in (l, l')"
                ax[(name, l, lp, m)] = (s, f"{lp}{l}{m}")
            continue
        assert A
        if m == 0:
            assert not B
            w(f"    const float2 A{l}{lp}{m} = {hsum(A)};", PHASES[2])
        else:
            # m >= 1: the (u+, w) 2x2 block [[A, s beta], [-s beta, A]] has eigenvectors (1, +-i) and eigenvalues
            # A +- i s beta; halved here because y'+ = (z+ + z-), z+- = E+- g+- with g+- = u'+ -+ i w'
            assert B
            Ah = [(p, 0.5 * cc) for (p, cc) in A]
            Bh = [(p, 0.5 * cc) for (p, cc) in B]
            w(f"    const float2 A{l}{lp}{m} = {hsum(Ah)};", PHASES[2])
            w(f"    const float2 E{l}{lp}{m}a = {hsum(Bh, f'A{l}{lp}{m}', True)};", PHASES[2])
            if len(Bh) == 1:
                w(f"    const float2 E{l}{lp}{m}b = {hsum([(p, -cc) for (p, cc) in Bh], f'A{l}{lp}{m}', True)};", PHASES[2])
            else:
                w(f"    const float2 E{l}{lp}{m}b = fma2(bc2(2.0f), A{l}{lp}{m}, neg2(E{l}{lp}{m}a));", PHASES[2])
        ax[("A", l, lp, m)] = (1, f"{l}{lp}{m}")
        ax[("B", l, lp, m)] = (1, f"{l}{lp}{m}") if B else (0, None)

    def rsum(terms, seed=None):
        """seed + sum of (sign, var, x): real coefficient times packed complex; var None means the constant 1"""
        plain = [(s, x) for (s, v, x) in terms if v is None and s != 0]
        mult = [(s, v, x) for (s, v, x) in terms if v is not None and s != 0]
        e = seed
        for (s, v, x) in mult:
            e = f"mul2({bcast(s, v)}, {x})" if e is None else f"fma2({bcast(s, v)}, {x}, {e})"
        for (s, x) in plain:
            if e is None:
                e = x if s > 0 else f"neg2({x})"
            else:
                e = f"add2({e}, {x})" if s > 0 else f"sub2({e}, {x})"
        assert e is not None
        return e

    def cchain(terms, seed=None):
        """seed + sum of (sign, complex coefficient variable, x): two packed instructions per term"""
        e = seed
        for (s, k, x) in terms:
            kk = k if s > 0 else f"neg2({k})"
            e = f"cmul2({kk}, {x})" if e is None else f"cfma2({kk}, {x}, {e})"
        return e

    tau_lines = []
    for ts in (0, 1):
        tsign = 1 if ts == 0 else -1
        tau_start = len(out)
        w(f"    {{ // tau block {'S = (1+2)/sqrt2' if ts == 0 else 'A = (1-2)/sqrt2'}")
        # (1) load + z-rotation (real plane rotation of (u+_m, w_m)); (2) y-rotation, with g+- = u'+ -+ i w' formed
        # inside the chains: g+ seeded with -i w', g- = g+ + 2 i w'
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            w(f"      const float2 zp{l}_0 = bload({o});")
            for m in range(1, l + 1):
                w(f"      const float2 bp{l}_{m} = bload({o + 2 * m - 1}), bw{l}_{m} = bload({o + 2 * m});")
                w(f"      const float2 zp{l}_{m} = fma2(bc2(cm[{m}]), bp{l}_{m}, mul2(bc2(sm[{m}]), bw{l}_{m}));", PHASES[3])
                w(f"      const float2 zw{l}_{m} = fma2(bc2(cm[{m}]), bw{l}_{m}, mul2(bc2(-sm[{m}]), bp{l}_{m}));", PHASES[3])
            terms = [(*R[("p", l, 0, m)], f"zp{l}_{m}") for m in range(0, l + 1)]
            w(f"      const float2 up{l}_0 = {rsum(terms)};", PHASES[4])
            for mt in range(1, l + 1):
                terms = [(*R[("m", l, mt - 1, m - 1)], f"zw{l}_{m}") for m in range(1, l + 1)]
                w(f"      const float2 uw{l}_{mt} = {rsum(terms)};", PHASES[4])
                terms = [(*R[("p", l, mt, m)], f"zp{l}_{m}") for m in range(0, l + 1)]
                w(f"      const float2 gp{l}_{mt} = {rsum(terms, f'nimul2(uw{l}_{mt})')};", PHASES[4])
                w(f"      const float2 gm{l}_{mt} = fma2(bc2(2.0f), imul2(uw{l}_{mt}), gp{l}_{mt});", PHASES[4])
        # (3) axial translation.  m = 0: y'+ = A u'+.  m >= 1: z+ = sum E g+, y'+ = z+ + sum E' g-, y'w = i (2 z+ - y'+)
        for l in range(1, lmax + 1):
            terms = []
            for lp in range(1, lmax + 1):
                sa, va = ax[("A", l, lp, 0)]
                if sa:
                    terms.append((sa, "A" + va, f"up{lp}_0"))
            assert terms
            w(f"      const float2 yp{l}_0 = {cchain(terms)};", PHASES[5])
            for mt in range(1, l + 1):
                tp, tm = [], []
                for lp in range(mt, lmax + 1):
                    sa, va = ax[("A", l, lp, mt)]
                    sb, vb = ax[("B", l, lp, mt)]
                    assert sa and sb and va == vb
                    plus, minus = ("a", "b") if sa * sb * tsign > 0 else ("b", "a")
                    tp.append((sa, f"E{va}{plus}", f"gp{lp}_{mt}"))
                    tm.append((sa, f"E{va}{minus}", f"gm{lp}_{mt}"))
                w(f"      const float2 zq{l}_{mt} = {cchain(tp)};", PHASES[5])
                w(f"      const float2 yp{l}_{mt} = {cchain(tm, f'zq{l}_{mt}')};", PHASES[5])
                w(f"      const float2 yw{l}_{mt} = fma2(bc2(2.0f), imul2(zq{l}_{mt}), nimul2(yp{l}_{mt}));", PHASES[5])
        # (4) rotate back (transposes), (5) z-rotate back and accumulate; every chain that ends in an accumulator
        # starts from it
        for l in range(1, lmax + 1):
            o = ts * H + (l - 1) * (l + 1)
            for m in range(0, l + 1):
                terms = [(*R[("p", l, mt, m)], f"yp{l}_{mt}") for mt in range(0, l + 1)]
                if m == 0:
                    w(f"      yacc.put({o}, {rsum(terms, f'yacc.get({o})')});", PHASES[6])
                else:
                    w(f"      const float2 vp{l}_{m} = {rsum(terms)};", PHASES[6])
            for m in range(1, l + 1):
                terms = [(*R[("m", l, mt - 1, m - 1)], f"yw{l}_{mt}") for mt in range(1, l + 1)]
                w(f"      const float2 vw{l}_{m} = {rsum(terms)};", PHASES[6])
            for m in range(1, l + 1):
                # y+ += c v+ - s vw ;  yw += s v+ + c vw
                qp, qw = o + 2 * m - 1, o + 2 * m
                w(f"      yacc.put({qp}, fma2(bc2(-sm[{m}]), vw{l}_{m}, fma2(bc2(cm[{m}]), vp{l}_{m}, yacc.get({qp}))));", PHASES[7])
                w(f"      yacc.put({qw}, fma2(bc2(cm[{m}]), vw{l}_{m}, fma2(bc2(sm[{m}]), vp{l}_{m}, yacc.get({qw}))));", PHASES[7])
        w("    }")
        tau_lines.append(out[tau_start:])
        del out[tau_start:]
    if interleave:       # the two tau blocks line by line (same coefficients back to back), variables suffixed s / a
        blk = [[_TAUVAR.sub(lambda mo, x=x: mo.group(1) + mo.group(2) + x, ln) for ln in lines[1:-1]]
               for lines, x in zip(tau_lines, "sa")]
        assert len(blk[0]) == len(blk[1])
        out.append("    { // tau blocks S = (1+2)/sqrt2 and A = (1-2)/sqrt2, interleaved")
        for ls, la in zip(*blk):
            out.extend([ls, la])
        out.append("    }")
    else:
        out.extend(tau_lines[0] + tau_lines[1])
    w("  }")
    w("};")
    outdir = outdir or os.path.join(HERE, "generated")
    os.makedirs(outdir, exist_ok=True)
    path = os.path.join(outdir, f"coupling_pk_lmax{lmax}.inc")
    with open(path, "w") as f:
        f.write("\n".join(out) + "\n")
    tot = [sum(c[k] for c in counts.values()) for k in range(4)]
    print(f"lmax={lmax}: {len(ent.defs)} unique rotation entries; packed FMA/MUL/ADD {tot[0]}/{tot[1]}/{tot[2]}, "
          f"scalar {tot[3]} (+ geometry and h_p recurrence in pair_math.cuh) -> {path}")
    if table is not None:
        table.append((lmax, counts))


def phase_table(tables):
    """markdown: per-phase source-level operation counts of the generated bodies"""
    lines = []
    for lmax, counts in tables:
        lines.append(f"\nlmax = {lmax} (both tau blocks; packed = FFMA2 / FMUL2 / FADD2 instructions, scalar = FFMA / FMUL)\n")
        lines.append("| phase | packed FMA | packed MUL | packed ADD | scalar |")
        lines.append("|---|---|---|---|---|")
        tot = [0, 0, 0, 0]
        for ph in PHASES:
            c = counts[ph]
            lines.append(f"| {ph} | {c[0]} | {c[1]} | {c[2]} | {c[3]} |")
            tot = [a + b for a, b in zip(tot, c)]
        lines.append(f"| **generated body** | {tot[0]} | {tot[1]} | {tot[2]} | {tot[3]} |")
    return "\n".join(lines)


if __name__ == "__main__":
    args = [a for a in sys.argv[1:] if not a.startswith("--")]
    tables = [] if "--table" in sys.argv else None
    for L in ([int(a) for a in args] or [1, 2, 3, 4, 5]):
        emit(L, table=tables)
    if tables is not None:
        print(phase_table(tables))
