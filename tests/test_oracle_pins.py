"""Pins of the FP64 oracle (oracle/) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the oracle
(a dropped term, a wrong sign or index, a transposed operand, a wrong normalisation) fails at least one.
Pin numbers follow DESIGN.md section 3 / SURVEY.md section 8(c).
"""
import itertools

import numpy as np
import pytest
from scipy.special import lpmv, spherical_jn, spherical_yn

import oracle as o

K = 2.0 * np.pi / 550.0          # 1/nm, background wavenumber of every config


def _rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b))


# --------------------------------------------------------------------------- P9 Wigner-3j
def test_p9_wigner3j_matches_sympy_exact():
    from sympy import N as symN
    from sympy.physics.wigner import wigner_3j
    rng = np.random.default_rng(9)
    cases = [(1, 1, 2, 1, -1, 0), (3, 3, 6, 3, -3, 0), (4, 4, 8, -2, 1, 1), (2, 3, 4, 0, 0, 0), (3, 4, 1, 2, -3, 1)]
    for _ in range(60):
        j1, j2 = rng.integers(1, 9, 2)
        j3 = rng.integers(abs(j1 - j2), j1 + j2 + 1)
        m1 = rng.integers(-j1, j1 + 1); m2 = rng.integers(-j2, j2 + 1)
        cases.append((int(j1), int(j2), int(j3), int(m1), int(m2), int(-m1 - m2)))
    for c in cases:
        assert o.wigner3j(*c) == pytest.approx(float(symN(wigner_3j(*c), 30)), abs=1e-14), c


def test_p9_wigner3j_orthogonality():
    # sum_{m1,m2} (2 j3 + 1) (j1 j2 j3; m1 m2 m3)(j1 j2 j3'; m1 m2 m3') = delta_{j3 j3'} delta_{m3 m3'}
    j1, j2 = 3, 4
    for j3, j3p in itertools.product(range(1, 8), repeat=2):
        for m3 in range(-min(j3, j3p), min(j3, j3p) + 1):
            s = sum((2 * j3 + 1) * o.wigner3j(j1, j2, j3, m1, m2, m3) * o.wigner3j(j1, j2, j3p, m1, m2, m3)
                    for m1 in range(-j1, j1 + 1) for m2 in range(-j2, j2 + 1))
            assert s == pytest.approx(1.0 if j3 == j3p else 0.0, abs=1e-13)


def test_a5_real_b5_imaginary_and_selection_rules():
    # a5 purely real, non-zero only for l+l'+p even; b5 purely imaginary, only for l+l'+p odd
    na = nb = 0
    for l, lp in itertools.product(range(1, 4), repeat=2):
        for m, mp in itertools.product(range(-l, l + 1), range(-lp, lp + 1)):
            for p in range(0, 7):
                a, b = o.a5(l, m, lp, mp, p), o.b5(l, m, lp, mp, p)
                assert abs(a.imag) < 1e-15 and abs(b.real) < 1e-15
                if (l + lp + p) % 2 == 1:
                    assert abs(a) < 1e-15
                else:
                    assert abs(b) < 1e-15
                na += abs(a) > 1e-14; nb += abs(b) > 1e-14
    assert (na, nb) == (461, 292)        # exact term counts quoted in SURVEY.md section 8(a) for lmax = 3


# --------------------------------------------------------------------------- Legendre / radial functions
def test_legendre_normalisation_and_library_agreement():
    x = np.linspace(-0.99, 0.99, 41)
    for l in range(0, 9):
        for m in range(0, l + 1):
            ours = np.array([o.legendre_normalized(l, m, xi) for xi in x])
            from math import factorial
            nrm = np.sqrt((2 * l + 1) / 2 * factorial(l - m) / factorial(l + m))
            assert np.allclose(ours, nrm * (-1) ** m * lpmv(m, l, x), atol=1e-12)      # SciPy carries the CS phase
    # orthonormality  int_{-1}^{1} P_l^m P_l'^m dx = delta_ll'   ("normalized")
    xs, ws = np.polynomial.legendre.leggauss(40)
    for m in range(0, 4):
        for l, lp in itertools.product(range(m, 7), repeat=2):
            v = sum(w * o.legendre_normalized(l, m, xx) * o.legendre_normalized(lp, m, xx) for xx, w in zip(xs, ws))
            assert v == pytest.approx(1.0 if l == lp else 0.0, abs=1e-12)
    assert o.legendre_normalized(0, 0, 0.3) == pytest.approx(1 / np.sqrt(2))
    assert o.legendre_normalized(1, 1, 0.6) == pytest.approx(np.sqrt(3) / 2 * 0.8)     # + sqrt(3)/2 sin(theta)


def test_python_legendre_pi_tau_against_cpp_and_finite_differences():
    th = np.linspace(0.2, 2.9, 17)
    P, pi, tau = o.legendre_pi_tau(6, np.cos(th), np.sin(th))
    h = 1e-6
    Pp, _, _ = o.legendre_pi_tau(6, np.cos(th + h), np.sin(th + h))
    Pm, _, _ = o.legendre_pi_tau(6, np.cos(th - h), np.sin(th - h))
    for l in range(1, 7):
        for m in range(0, l + 1):
            cpp = np.array([o.legendre_normalized(l, m, c) for c in np.cos(th)])
            assert np.allclose(P[(l, m)], cpp, atol=1e-13)
            if m > 0:
                assert np.allclose(pi[(l, m)] * np.sin(th), cpp, atol=1e-13)
            assert np.allclose(tau[(l, m)], (Pp[(l, m)] - Pm[(l, m)]) / (2 * h), atol=1e-7)


def test_radial_is_hankel_first_kind():
    for p in range(0, 9):
        for x in (2.3, 7.7, 150.0):
            h = o.radial(3, p, x)
            assert h.real == pytest.approx(spherical_jn(p, x), rel=1e-12, abs=1e-15)
            assert h.imag == pytest.approx(spherical_yn(p, x), rel=1e-12, abs=1e-15)
    x = 5.0   # h_0^(1)(x) = -i e^{ix} / x
    assert o.radial(3, 0, x) == pytest.approx(-1j * np.exp(1j * x) / x, abs=1e-14)


def test_radial_large_argument():
    """Beyond x = 8000 the oracle leaves libstdc++ (which throws near 1.5e4) for the closed forms of order 0, 1 and the
    upward recurrence: against SciPy on both sides of the switch, and continuous across it."""
    for x in (7999.5, 8000.5, 1.2e4, 2.0e4, 5.3e4):
        for p in range(0, 11):
            h = o.radial(3, p, x)
            ref = spherical_jn(p, x) + 1j * spherical_yn(p, x)
            assert abs(h - ref) <= 2e-9 * abs(ref), (x, p)
            assert o.radial(1, p, x).real == pytest.approx(spherical_jn(p, x), abs=2e-9 * abs(ref))
            assert o.radial(2, p, x).real == pytest.approx(spherical_yn(p, x), abs=2e-9 * abs(ref))
    # a block far away is what the far-field limit says: W ~ e^{ikd}/(kd) times an angular factor, |W| ~ 1/kd
    d1, d2 = np.array([0.0, 0.0, 0.7e6]), np.array([0.0, 0.0, 1.4e6])
    w1, w2 = o.coupling_block(2, K, d1), o.coupling_block(2, K, d2)
    assert np.linalg.norm(w2) / np.linalg.norm(w1) == pytest.approx(0.5, rel=1e-3)


# --------------------------------------------------------------------------- P1 addition theorem (A.5)
@pytest.mark.parametrize("n", [(1, 1, 0), (1, 1, -1), (2, 1, 1), (1, 2, -2), (2, 2, 1), (1, 3, 3), (2, 3, -2), (2, 3, 0),
                               (1, 4, -3), (2, 4, 4)])
def test_p1_addition_theorem_brute_force(n):
    # Psi^(3)_n(r + d) = sum_{n'} A_{nn'}(d) Psi^(1)_{n'}(r), |r| < |d|   (A.5)
    d = 2.7 / K * np.array([0.48, -0.62, 0.62]) / np.linalg.norm([0.48, -0.62, 0.62])
    r = 0.3 / K * np.array([[0.3, 0.5, -0.81], [-0.7, 0.1, 0.2], [0.05, -0.6, 0.79]])
    r = r / np.linalg.norm(r, axis=1, keepdims=True) * 0.3 / K
    lhs = o.svwf(3, n[0], n[1], n[2], K, r + d)
    rhs = np.zeros_like(lhs)
    for taup in (1, 2):
        for lp in range(1, 15):
            for mp in range(-lp, lp + 1):
                rhs += o.translation_A(n, (taup, lp, mp), K, d) * o.svwf(1, taup, lp, mp, K, r)
    assert _rel(rhs, lhs) < 1e-8


def test_p1_wrong_conventions_fail():
    # the check above has teeth: flipping the azimuthal sign, or dropping the normalisation of P, breaks it
    n = (2, 2, 1)
    d = 2.7 / K * np.array([0.48, -0.62, 0.62]) / np.linalg.norm([0.48, -0.62, 0.62])
    r = 0.3 / K * np.array([[0.3, 0.5, -0.81]])
    lhs = o.svwf(3, *n, K, r + d)
    rhs = np.zeros_like(lhs)
    dflip = d * np.array([1, -1, 1])           # phi_d -> -phi_d
    for taup in (1, 2):
        for lp in range(1, 13):
            for mp in range(-lp, lp + 1):
                rhs += o.translation_A(n, (taup, lp, mp), K, dflip) * o.svwf(1, taup, lp, mp, K, r)
    assert _rel(rhs, lhs) > 1e-2


# --------------------------------------------------------------------------- P2 physical form of eq. (7)
def test_p2_coupling_block_reexpands_emitter_field_about_receiver():
    # field of emitter i' with unit coefficient n', Psi^(3)_{n'}(r - r_i'), equals sum_n W_{nn'} Psi^(1)_n(r - r_i)
    # near r_i: this fixes the direction of d (R7), the transposition of eq. (7) and the sign of the phase (R6).
    L = 10
    ri = np.array([230.0, 40.0, -60.0]); rip = np.array([0.0, 0.0, 0.0])
    W = o.coupling_block(L, K, ri - rip)
    pts = ri + 0.25 / K * np.array([[0.2, -0.5, 0.84], [-0.6, 0.64, 0.48], [0.1, 0.1, -0.99]])
    idx = o.multi_indices(L)
    for nprime in [(1, 1, 1), (2, 1, 0), (1, 2, -2), (2, 3, 3), (1, 3, -1), (2, 2, 1)]:
        lhs = o.svwf(3, *nprime, K, pts - rip)
        col = o.nindex(L, *nprime)
        rhs = sum(W[o.nindex(L, *n), col] * o.svwf(1, *n, K, pts - ri) for n in idx)
        assert _rel(rhs, lhs) < 1e-7


def test_cached_block_equals_term_by_term_translation_operator():
    d = np.array([-140.0, 95.0, 210.0])
    for lmax in (2, 3, 4):
        W = o.coupling_block(lmax, K, d)
        idx = o.multi_indices(lmax)
        ref = np.array([[o.translation_A(npr, n, K, d) for npr in idx] for n in idx])   # W_{nn'} = A_{n'n}
        assert np.max(np.abs(W - ref)) < 1e-13 * np.max(np.abs(ref))


# --------------------------------------------------------------------------- P3, P4, P4b structure
def test_p3_on_axis_pairs_are_diagonal_in_m():
    idx = o.multi_indices(3)
    for d in ([0, 0, 300.0], [0, 0, -450.0]):
        W = o.coupling_block(3, K, d)
        assert np.all(np.isfinite(W.view(np.float64)))
        for a, n in enumerate(idx):
            for b, npr in enumerate(idx):
                if n[2] != npr[2]:
                    assert W[a, b] == 0
        assert np.linalg.norm(W) > 1.0


def test_p4_parity_under_d_to_minus_d():
    # W^{i'i}_{nn'} = (-1)^{l+l'+tau+tau'} W^{ii'}_{nn'}
    idx = o.multi_indices(4)
    d = np.array([230.0, 40.0, -60.0])
    Wp, Wm = o.coupling_block(4, K, d), o.coupling_block(4, K, -d)
    sgn = np.array([[(-1) ** (n[1] + npr[1] + n[0] + npr[0]) for npr in idx] for n in idx])
    assert np.max(np.abs(Wm - sgn * Wp)) < 1e-13 * np.max(np.abs(Wp))


def test_p4b_tau_blocks_and_regular_part_hermitian():
    d = np.array([-310.0, 120.0, 75.0])
    for lmax in (3, 4):
        h = o.nmax_of(lmax) // 2
        W = o.coupling_block(lmax, K, d)
        assert np.array_equal(W[:h, :h], W[h:, h:]) and np.array_equal(W[:h, h:], W[h:, :h])
        for kind in (1, 2):   # Bessel part and Neumann part separately
            R, Rm = o.coupling_block(lmax, K, d, kind=kind), o.coupling_block(lmax, K, -d, kind=kind)
            assert np.max(np.abs(Rm - R.conj().T)) < 1e-13 * np.max(np.abs(R))


# --------------------------------------------------------------------------- P7 golden W entries
def test_p7_golden_coupling_entries(golden):
    g = golden("p7_w_entries.txt")
    W = o.coupling_block(3, K, (230.0, 40.0, -60.0))
    for key, v in g.items():
        if key.startswith("W_"):
            _, a, b = key.split("_")
            assert W[int(a), int(b)] == pytest.approx(complex(v[0], v[1]), rel=1e-13, abs=1e-15), key
    assert np.linalg.norm(W) == pytest.approx(g["normF"][0], rel=1e-13)


# --------------------------------------------------------------------------- P5, P6 single sphere -> Mie
def _bohren_huffman(l, x, m):
    """Textbook Mie coefficients a_l, b_l (Bohren & Huffman eq. 4.53) from Riccati-Bessel functions."""
    psi = lambda z: z * spherical_jn(l, z)
    dpsi = lambda z: spherical_jn(l, z) + z * spherical_jn(l, z, derivative=True)
    xi = lambda z: z * (spherical_jn(l, z) + 1j * spherical_yn(l, z))
    dxi = lambda z: (spherical_jn(l, z) + 1j * spherical_yn(l, z)) + z * (
        spherical_jn(l, z, derivative=True) + 1j * spherical_yn(l, z, derivative=True))
    a = (m * psi(m * x) * dpsi(x) - psi(x) * dpsi(m * x)) / (m * psi(m * x) * dxi(x) - xi(x) * dpsi(m * x))
    b = (psi(m * x) * dpsi(x) - m * psi(x) * dpsi(m * x)) / (psi(m * x) * dxi(x) - m * xi(x) * dpsi(m * x))
    return a, b


def test_p6_mie_golden_values_and_textbook_form(golden):
    g = golden("p6_mie_q.txt")
    Q = o.mie_q(3, K, [100.0], 1.52)
    for tau in (1, 2):
        for l in (1, 2, 3):
            v = g[f"Q_{tau}_{l}"]
            assert Q[0, tau - 1, l - 1] == pytest.approx(complex(v[0], v[1]), rel=2e-12)
    for ni in (1.52, 1.52 + 0.1j, 2.4 + 0.02j):
        Q = o.mie_q(4, K, [100.0, 83.0], ni)
        for i, R in enumerate((100.0, 83.0)):
            for l in range(1, 5):
                a, b = _bohren_huffman(l, K * R, ni)
                assert Q[i, 0, l - 1] == pytest.approx(-b, rel=1e-11)        # reading R11
                assert Q[i, 1, l - 1] == pytest.approx(-a, rel=1e-11)
    Q = o.mie_q(3, K, [100.0], 1.52)
    assert np.allclose(Q.real, -np.abs(Q) ** 2, rtol=1e-10, atol=1e-18)      # lossless sphere: Re Q = -|Q|^2


def test_p5_single_sphere_reduces_to_mie_series(golden):
    R, ni, lmax = 100.0, 1.52, 3
    pos = np.zeros((1, 3))
    q = o.mie_q(lmax, K, [R], ni)
    a_in = o.plane_wave_a_in(pos, K, lmax)
    b = o.solve_dense(pos, K, lmax, q, a_in)
    assert np.array_equal(b, o.rhs(q, lmax, a_in))                       # N = 1: W b = 0, b = T a_in
    assert np.all(o.coupling_matvec(pos, K, lmax, b) == 0)
    x = K * R
    ab = [_bohren_huffman(l, x, ni) for l in range(1, lmax + 1)]
    qext = 2 / x**2 * sum((2 * l + 1) * (a + bb).real for l, (a, bb) in enumerate(ab, start=1))
    qsca = 2 / x**2 * sum((2 * l + 1) * (abs(a) ** 2 + abs(bb) ** 2) for l, (a, bb) in enumerate(ab, start=1))
    geo = np.pi * R**2
    assert o.extinction_cross_section(K, a_in, b) / geo == pytest.approx(qext, rel=1e-12)
    assert o.scattering_cross_section(pos, K, lmax, b) / geo == pytest.approx(qsca, rel=1e-12)
    assert qext == pytest.approx(golden("p6_mie_q.txt")["Q_ext"][0], rel=1e-12)
    # Rayleigh limit x -> 0: Q_sca -> (8/3) x^4 |(n^2-1)/(n^2+2)|^2
    Rs = 2.0
    qs = o.mie_q(1, K, [Rs], ni)
    bs = o.rhs(qs, 1, o.plane_wave_a_in(pos, K, 1))
    xs = K * Rs
    assert o.scattering_cross_section(pos, K, 1, bs) / (np.pi * Rs**2) == pytest.approx(
        8 / 3 * xs**4 * abs((ni**2 - 1) / (ni**2 + 2)) ** 2, rel=2e-3)


# --------------------------------------------------------------------------- P10 plane-wave expansion (A.13)
@pytest.mark.parametrize("alpha,beta", [(0.0, 0.0), (0.7, 1.1), (-2.0, 2.6), (3.0, 0.4)])
@pytest.mark.parametrize("j", [1, 2])
def test_p10_plane_wave_expansion(alpha, beta, j):
    L = 16
    pts = 0.8 / K * np.array([[0.3, -0.4, 0.5], [-0.5, 0.2, -0.1], [0.0, 0.6, 0.3]])
    a = o.plane_wave_a_in(np.zeros((1, 3)), K, L, alpha, beta, j)[0]
    field = sum(a[o.nindex(L, *n)] * o.svwf(1, *n, K, pts) for n in o.multi_indices(L))
    assert _rel(field, o.pvwf(j, alpha, beta, K, pts)) < 1e-12


def test_plane_wave_normal_incidence_closed_form_and_centre_phase():
    # +z, x-polarised: a_(tau,l,m) = e^{ikz_i} (-i^{l+1}) sqrt(2l+1) delta_{|m|,1} (1 if tau = 2 else m)
    pos = np.array([[10.0, -20.0, 35.0], [400.0, 0.0, -120.0]])
    a = o.plane_wave_a_in(pos, K, 4)
    for i in range(2):
        for (tau, l, m) in o.multi_indices(4):
            want = 0.0
            if abs(m) == 1:
                want = np.exp(1j * K * pos[i, 2]) * (-(1j ** (l + 1))) * np.sqrt(2 * l + 1) * (1 if tau == 2 else m)
            assert a[i, o.nindex(4, tau, l, m)] == pytest.approx(want, abs=1e-13)
    # shifted-origin expansion reproduces the same global field
    pts = pos[1] + 0.5 / K * np.array([[0.3, 0.1, -0.2]])
    L = 14
    aL = o.plane_wave_a_in(pos, K, L)
    field = sum(aL[1, o.nindex(L, *n)] * o.svwf(1, *n, K, pts - pos[1]) for n in o.multi_indices(L))
    assert _rel(field, o.pvwf(2, 0.0, 0.0, K, pts)) < 1e-12


# --------------------------------------------------------------------------- P8 optical theorem
POS3 = np.array([[0.0, 0.0, 0.0], [230.0, 40.0, -60.0], [-80.0, 250.0, 150.0]])


def test_p8_optical_theorem_lossless_and_absorbing(golden):
    g = golden("p8_optical_theorem.txt")
    q = o.mie_q(3, K, [100.0] * 3, 1.52)
    a_in = o.plane_wave_a_in(POS3, K, 3)
    b = o.solve_dense(POS3, K, 3, q, a_in)
    cext, csca = o.extinction_cross_section(K, a_in, b), o.scattering_cross_section(POS3, K, 3, b)
    assert cext == pytest.approx(csca, rel=1e-12)
    assert cext == pytest.approx(g["C_ext_nm2"][0], rel=1e-11)
    for n in range(3):
        v = g[f"b_0_{n}"]
        assert b[0, n] == pytest.approx(complex(v[0], v[1]), rel=1e-9)
    qa = o.mie_q(3, K, [100.0] * 3, 1.52 + 0.1j)
    ba = o.solve_dense(POS3, K, 3, qa, a_in)
    cext_a, csca_a = o.extinction_cross_section(K, a_in, ba), o.scattering_cross_section(POS3, K, 3, ba)
    assert cext_a == pytest.approx(g["C_ext_abs_nm2"][0], rel=1e-5)
    assert csca_a == pytest.approx(g["C_sca_abs_nm2"][0], rel=1e-5)
    assert cext_a > csca_a                                                   # reading R10


# --------------------------------------------------------------------------- P11 brute force on tiny inputs
def test_p11_matvec_equals_dense_assembly_and_gmres_equals_lu():
    from paper_1706_02145_b200 import workloads as wl
    w = wl.scaled(wl.C2, 24)
    pos, rad = wl.positions(w)
    q = o.mie_q(w.lmax, w.k, rad, wl.N_SPHERE)
    b = wl.gaussian_coefficients(w.N, w.nmax, w.seed_b).astype(np.complex128)
    W = o.dense_coupling_matrix(pos, w.k, w.lmax)
    y = o.coupling_matvec(pos, w.k, w.lmax, b)
    assert _rel(y.reshape(-1), W @ b.reshape(-1)) < 1e-13
    sub = np.array([3, 17, 5], dtype=np.int64)
    assert np.array_equal(o.coupling_matvec(pos, w.k, w.lmax, b, receivers=sub), y[sub])
    M = o.dense_system_matrix(pos, w.k, w.lmax, q)
    assert _rel(o.system_matvec(pos, w.k, w.lmax, q, b).reshape(-1), M @ b.reshape(-1)) < 1e-13
    a_in = o.plane_wave_a_in(pos, w.k, w.lmax)
    x_lu = o.solve_dense(pos, w.k, w.lmax, q, a_in)
    x_it, info = o.solve_gmres(pos, w.k, w.lmax, q, a_in, rtol=1e-11, restart=40)
    assert info["rel_residual"] <= 1e-11
    assert _rel(x_it, x_lu) < 1e-9


# --------------------------------------------------------------------------- P13 block-diagonal preconditioner
def test_p13_preconditioner_limits_and_partition_brute_force():
    """PAPER.md:109-116.  (a) one cuboid holding every sphere: the preconditioner IS M^{-1} (dense LU of eq. 8);
    (b) cuboids so small that every sphere is alone: M_j = 1 (W^{ii} = 0), z = v; (c) the partition against a
    brute-force pairwise statement of "same cuboid"; (d) two clusters far apart cut between them: M z = v up to
    the weak far coupling, and exactly M_jj z_j = v_j block by block."""
    from paper_1706_02145_b200 import workloads as wl
    w = wl.scaled(wl.C2, 20)
    pos, rad = wl.positions(w)
    q = o.mie_q(w.lmax, w.k, rad, wl.N_SPHERE)
    n = o.nmax_of(w.lmax)
    v = wl.gaussian_coefficients(w.N, w.nmax, 77).astype(np.complex128)
    M = o.dense_system_matrix(pos, w.k, w.lmax, q)
    # (a)
    z = o.precond_apply(pos, w.k, w.lmax, q, [0.0, 0.0, 0.0], v)
    assert _rel(M @ z.reshape(-1), v.reshape(-1)) < 1e-11
    # (b)
    assert np.array_equal(o.precond_apply(pos, w.k, w.lmax, q, 1.0, v), v)
    # (c)
    edge = np.array([700.0, 900.0, 0.0])
    groups = o.cuboid_partition(pos, edge)
    label = np.empty(w.N, dtype=int)
    for j, idx in enumerate(groups):
        label[idx] = j
    assert sorted(np.concatenate(groups).tolist()) == list(range(w.N))
    lo = pos.min(axis=0)
    for i in range(w.N):
        for ip in range(w.N):
            same = all(edge[a] <= 0 or int((pos[i, a] - lo[a]) // edge[a]) == int((pos[ip, a] - lo[a]) // edge[a])
                       for a in range(3))
            assert same == (label[i] == label[ip])
    # (d)
    far = pos.copy()
    half = pos[:, 0] > np.median(pos[:, 0])
    far[half, 0] += 4.0e5                                      # second cluster 400 um away
    span = far[:, 0].max() - far[:, 0].min()
    gr = o.cuboid_partition(far, [0.6 * span, 0.0, 0.0])
    assert len(gr) == 2 and set(gr[1].tolist()) == set(np.nonzero(half)[0].tolist())
    Mf = o.dense_system_matrix(far, w.k, w.lmax, q)
    zf = o.precond_apply(far, w.k, w.lmax, q, [0.6 * span, 0.0, 0.0], v)
    for idx in gr:
        rows = (idx[:, None] * n + np.arange(n)[None, :]).reshape(-1)
        assert _rel(Mf[np.ix_(rows, rows)] @ zf[idx].reshape(-1), v[idx].reshape(-1)) < 1e-11
    assert _rel(Mf @ zf.reshape(-1), v.reshape(-1)) < 1e-2      # coupling ~ 1/(k d) across 400 um


# --------------------------------------------------------------------------- P14 far field (A.12, D.1-D.3)
def test_p14_far_field_power_equals_scattering_cross_section(golden):
    """The flux of the plane-wave amplitudes g_j (A.12 about every sphere, D.2) over the full sphere of directions
    equals C_sca of P8 (golden value, PAPER-derived; and the oracle's regular-translation formula): fixes the 1/2pi of
    (A.12), the prefactor of (D.2)-(D.3), the sign of the origin-shift phase and the roles of B_n1, B_n2.  A rigid
    shift of the cluster multiplies g by a pure phase; a single sphere with one coefficient gives |B_nj| / 2 pi."""
    g8 = golden("p8_optical_theorem.txt")
    q = o.mie_q(3, K, [100.0] * 3, 1.52)
    a_in = o.plane_wave_a_in(POS3, K, 3)
    b = o.solve_dense(POS3, K, 3, q, a_in)
    xb, wb = np.polynomial.legendre.leggauss(40)
    na = 80
    A, B = np.meshgrid(2 * np.pi * np.arange(na) / na, np.arccos(xb), indexing="ij")
    W = np.broadcast_to(wb[None, :] * 2 * np.pi / na, A.shape)
    g = o.far_field_amplitude(POS3, K, 3, b, A.ravel(), B.ravel())
    csca = o.scattered_power_cross_section(K, g, W.ravel())
    assert csca == pytest.approx(g8["C_sca_nm2"][0], rel=1e-9)
    assert csca == pytest.approx(o.scattering_cross_section(POS3, K, 3, b), rel=1e-9)
    shift = np.array([310.0, -120.0, 75.0])
    gs = o.far_field_amplitude(POS3 + shift, K, 3, b, A.ravel()[:50], B.ravel()[:50])
    kv = K * np.stack([np.sin(B.ravel()[:50]) * np.cos(A.ravel()[:50]), np.sin(B.ravel()[:50]) * np.sin(A.ravel()[:50]),
                       np.cos(B.ravel()[:50])], axis=1)
    assert np.allclose(gs, g[:50] * np.exp(-1j * (kv @ shift))[:, None], rtol=1e-12, atol=1e-15)
    e = np.zeros((1, o.nmax_of(3)), dtype=np.complex128)
    n = o.nindex(3, 2, 2, -1)
    e[0, n] = 1.0
    g1 = o.far_field_amplitude(np.zeros((1, 3)), K, 3, e, [0.7], [1.1])
    for j in (1, 2):
        assert g1[0, j - 1] == pytest.approx(o.plane_wave_B(3, 1.1, j)[n] * np.exp(-1j * 0.7) / (2 * np.pi), rel=1e-13)


# --------------------------------------------------------------------------- P15 Gaussian beam (Appendix C)
def test_p15_gaussian_beam_coefficients():
    """(C.8) with the analytic azimuthal integral (C.7) against the angular spectrum (C.4) integrated by brute force
    with the exact phase e^{ik.(r_i - r_G)} (fixes reading R20 of the garbled (C.5), the Bessel identity, the orders
    |m -+ 1| and the factor k^2 w^2 / pi); the field rebuilt from the coefficients near the waist against the Gaussian
    profile of (C.1) (fixes k^2 w^2 / 4 pi and the polarisation vector; paraxial, so to ~1/(kw)^2); and the beam power:
    the flux of g of (D.4) equals (D.5)."""
    pos = np.array([[0.0, 0.0, 0.0], [230.0, 40.0, -60.0], [-800.0, 1250.0, 150.0], [1500.0, -300.0, -200.0]])
    w, rG, aG = 2000.0, np.array([100.0, -50.0, 30.0]), 0.4
    a = o.gaussian_beam_a_in(pos, K, 3, w, rG, aG, n_beta=300)
    a_bf = o.gaussian_beam_a_in_brute_force(pos, K, 3, w, rG, aG)
    assert np.max(np.abs(a - a_bf)) <= 1e-12 * np.max(np.abs(a))
    for r in (np.array([[30.0, -20.0, 30.0]]), np.array([[-15.0, 25.0, 30.0]])):
        E = np.zeros(3, dtype=np.complex128)
        for n, (tau, l, m) in enumerate(o.multi_indices(3)):
            E += a[0, n] * o.svwf(1, tau, l, m, K, r - pos[0:1])[0]
        rho2 = np.sum((r[0, :2] - rG[:2]) ** 2)
        ref = np.exp(-rho2 / w**2) * np.array([-np.sin(aG), np.cos(aG), 0.0])
        assert np.max(np.abs(E - ref)) <= 6e-3
    xb, wb = np.polynomial.legendre.leggauss(400)
    beta, wbeta = (xb + 1.0) * np.pi / 4.0, wb * np.pi / 4.0
    na = 16
    A, B = np.meshgrid(2 * np.pi * np.arange(na) / na, beta, indexing="ij")
    W = np.broadcast_to((wbeta * np.sin(beta))[None, :] * 2 * np.pi / na, A.shape)
    g = o.gaussian_beam_g(K, w, rG, A.ravel(), B.ravel(), aG)
    flux = np.sum(W.ravel()[:, None] * np.abs(g) ** 2)                      # int sum_j |g_j|^2 sin(beta) d(beta) d(alpha)
    d5 = K**4 * w**4 / (8 * np.pi) * np.sum(wbeta * np.sin(beta) * np.cos(beta) ** 2 * np.exp(-w * w * K * K * np.sin(beta) ** 2 / 2))
    assert flux == pytest.approx(d5, rel=1e-12)                             # (D.5) / (2 pi^2 / (omega k mu_0))


# --------------------------------------------------------------------------- P16 near field (eq. 3)
def test_p16_scattered_field_is_consistent_with_far_field_and_translation():
    """scattered_field() sums svwf() (pinned by P1, P2) over spheres.  Independent checks of the sum: (a) far from the
    cluster it tends to the spherical wave of the plane-wave amplitudes g_j of P14 (A.12 evaluated by stationary phase:
    E -> -2 pi i e^{ikr}/(kr) sum_j g_j e_j), which ties eq. (3) to (A.12)/(A.14) including the per-sphere phase;
    (b) one sphere's outgoing field re-expanded about a second origin with the oracle's W block (eq. 7) gives the
    same field near that origin."""
    rng = np.random.default_rng(5)
    b = rng.normal(size=(3, 30)) + 1j * rng.normal(size=(3, 30))
    al, be = np.array([0.3, 2.0, 4.4]), np.array([0.5, 1.7, 2.6])
    rhat = np.stack([np.sin(be) * np.cos(al), np.sin(be) * np.sin(al), np.cos(be)], axis=1)
    R = 5.0e7                                                    # k R ~ 5.7e5: far field
    E = o.scattered_field(POS3, K, 3, b, R * rhat)
    g = o.far_field_amplitude(POS3, K, 3, b, al, be)
    e_al = np.stack([-np.sin(al), np.cos(al), np.zeros(3)], axis=1)
    e_be = np.stack([np.cos(be) * np.cos(al), np.cos(be) * np.sin(al), -np.sin(be)], axis=1)
    Eff = (-2j * np.pi * np.exp(1j * K * R) / (K * R))[..., None] * (g[:, 0:1] * e_al + g[:, 1:2] * e_be)
    assert np.max(np.abs(E - Eff)) <= 1e-4 * np.max(np.abs(Eff))
    # (b)
    d = POS3[1] - POS3[0]
    b0 = np.zeros((1, 30), dtype=np.complex128)
    b0[0] = b[0]
    pts = POS3[1][None, :] + np.array([[6.0, -3.5, 4.5], [-2.5, 7.0, 1.5]])
    E_direct = o.scattered_field(POS3[0:1], K, 3, b0, pts)
    a_loc = o.coupling_block(3, K, d) @ b[0]                      # regular coefficients about sphere 1, lmax = 3
    E_loc = np.zeros((2, 3), dtype=np.complex128)
    for n, (tau, l, m) in enumerate(o.multi_indices(3)):
        E_loc += a_loc[n] * o.svwf(1, tau, l, m, K, pts - POS3[1][None, :])
    assert np.max(np.abs(E_loc - E_direct)) <= 5e-4 * np.max(np.abs(E_direct))     # truncation of the regular series at l = 3
