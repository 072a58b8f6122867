"""CELES oracle (Python side) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

FP64, CPU, plain.  Each function cites the passage of PAPER.md it restates.  The N^2 coupling
sum itself lives in ``celes_oracle.cpp`` (same directory) and is reached through ctypes; this
file adds what surrounds it on the hot path: the sphere T-matrix (B.1-B.3), the system
operator of eqs. (8)-(9), the plane-wave right-hand side (A.13-A.14), a reference solve, the
block-diagonal preconditioner of PAPER.md:109-116 (cuboid partition, block-by-block dense solve), the far-field
amplitudes of (A.12)/(D.1)-(D.3), the Gaussian beam of Appendix C, and
the SVWF / PVWF evaluators (A.2, A.4) that the pins in tests/test_oracle_pins.py use for the
brute-force addition-theorem check.

Nothing in here imports, reads or shares anything with ``paper_1706_02145_b200/``.
Pins: see tests/test_oracle_pins.py (P1-P11, P13-P16 of DESIGN.md).  Nothing is "parity unpinned".
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np
from scipy.special import spherical_jn, spherical_yn

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "celes_oracle.cpp")
_SO = os.path.join(_HERE, "libceles_oracle.so")
_LIB = None
LAST_THREADS = 0  # OpenMP threads the last coupling_matvec call used


def build(force: bool = False) -> str:
    """Compile celes_oracle.cpp into libceles_oracle.so (g++ -O3 -march=native -fopenmp)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _SO]
        subprocess.run(cmd, check=True)
    return _SO


def _lib():
    global _LIB
    if _LIB is None:
        build()
        L = ctypes.CDLL(_SO)
        i, d, p = ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        L.oracle_wigner3j.restype = d
        L.oracle_wigner3j.argtypes = [i] * 6
        L.oracle_a5.argtypes = [i] * 5 + [p]
        L.oracle_b5.argtypes = [i] * 5 + [p]
        L.oracle_legendre_normalized.restype = d
        L.oracle_legendre_normalized.argtypes = [i, i, d]
        L.oracle_radial.argtypes = [i, i, d, p]
        L.oracle_translation_A.argtypes = [i] * 6 + [d] * 4 + [i, p]
        L.oracle_coupling_block.argtypes = [i, d, d, d, d, i, p]
        L.oracle_coupling_matvec.restype = i
        L.oracle_coupling_matvec.argtypes = [i, i, d, p, p, i, p, p, i]
        _LIB = L
    return _LIB


# ----------------------------------------------------------------------------- indices
def nmax_of(lmax: int) -> int:
    """n_max = 2 lmax (lmax + 2): tau in {1,2}, l = 1..lmax, m = -l..l."""
    return 2 * lmax * (lmax + 2)


def nindex(lmax: int, tau: int, l: int, m: int) -> int:
    """0-based multi-index, reading R1: tau outermost, then l, then m ascending."""
    return (tau - 1) * lmax * (lmax + 2) + (l - 1) * (l + 1) + (m + l)


def multi_indices(lmax: int):
    """List of (tau, l, m) in the order of nindex."""
    return [(tau, l, m) for tau in (1, 2) for l in range(1, lmax + 1) for m in range(-l, l + 1)]


# ----------------------------------------------------------------------------- thin ctypes wrappers
def _c2():
    return (ctypes.c_double * 2)()


def wigner3j(j1, j2, j3, m1, m2, m3) -> float:
    return _lib().oracle_wigner3j(j1, j2, j3, m1, m2, m3)


def a5(l, m, lp, mp, p) -> complex:
    """(A.9)-(A.10)."""
    o = _c2(); _lib().oracle_a5(l, m, lp, mp, p, o); return complex(o[0], o[1])


def b5(l, m, lp, mp, p) -> complex:
    """(A.11)."""
    o = _c2(); _lib().oracle_b5(l, m, lp, mp, p, o); return complex(o[0], o[1])


def legendre_normalized(l, m, x) -> float:
    """Normalised P_l^m(x) of PAPER.md:215 (reading R2), from std::assoc_legendre."""
    return _lib().oracle_legendre_normalized(l, m, float(x))


def radial(kind, p, x) -> complex:
    """z_p(x): kind 3 -> h_p^(1), 1 -> j_p, 2 -> y_p."""
    o = _c2(); _lib().oracle_radial(kind, p, float(x), o); return complex(o[0], o[1])


def translation_A(n, nprime, k, d, kind=3) -> complex:
    """A_{nn'}(d) of (A.6)-(A.8); n, n' = (tau, l, m) tuples; nothing cached."""
    o = _c2()
    _lib().oracle_translation_A(n[0], n[1], n[2], nprime[0], nprime[1], nprime[2], float(k),
                                float(d[0]), float(d[1]), float(d[2]), kind, o)
    return complex(o[0], o[1])


def coupling_block(lmax, k, d, kind=3) -> np.ndarray:
    """W^{ii'} for d = r_i - r_i' (eq. 7): [n, n'] complex128."""
    n = nmax_of(lmax)
    W = np.empty((n, n), dtype=np.complex128)
    _lib().oracle_coupling_block(lmax, float(k), float(d[0]), float(d[1]), float(d[2]), kind,
                                 W.ctypes.data_as(ctypes.c_void_p))
    return W


def coupling_matvec(pos, k, lmax, b, receivers=None, kind=3) -> np.ndarray:
    """y^i_n = sum_{i'!=i} sum_{n'} W^{ii'}_{nn'} b^{i'}_{n'} (eq. 6) for the receivers
    listed (default: all).  pos [N,3] float64; b [N,nmax] complex; returns [n_recv,nmax] complex128."""
    global LAST_THREADS
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    N = pos.shape[0]
    n = nmax_of(lmax)
    b = np.ascontiguousarray(np.asarray(b).reshape(N, n), dtype=np.complex128)
    recv = np.arange(N, dtype=np.int64) if receivers is None else np.ascontiguousarray(receivers, dtype=np.int64)
    y = np.zeros((recv.shape[0], n), dtype=np.complex128)
    LAST_THREADS = _lib().oracle_coupling_matvec(
        N, lmax, float(k), pos.ctypes.data_as(ctypes.c_void_p), b.ctypes.data_as(ctypes.c_void_p),
        recv.shape[0], recv.ctypes.data_as(ctypes.c_void_p), y.ctypes.data_as(ctypes.c_void_p), kind)
    return y


# ----------------------------------------------------------------------------- T-matrix (Appendix B)
def _d_xz(z, x, deriv):
    """d/dx (x z_l(x)) = z_l(x) + x z_l'(x)."""
    return z + x * deriv


def mie_q(lmax, k, radii, n_sphere, n0=1.0) -> np.ndarray:
    """Q^i_{tau,l} of (B.2)-(B.3).  k: background wavenumber; k_i = (n_i/n0) k.
    Returns [N, 2, lmax] complex128 (index [i, tau-1, l-1])."""
    radii = np.atleast_1d(np.asarray(radii, dtype=np.float64))
    n_sphere = np.broadcast_to(np.asarray(n_sphere, dtype=np.complex128), radii.shape)
    Q = np.empty((radii.shape[0], 2, lmax), dtype=np.complex128)
    for i, (R, ni) in enumerate(zip(radii, n_sphere)):
        ki = ni / n0 * k
        x, xi = k * R, ki * R                       # kR_i and k_i R_i
        for l in range(1, lmax + 1):
            j_x, dj_x = spherical_jn(l, x), spherical_jn(l, x, derivative=True)
            y_x, dy_x = spherical_yn(l, x), spherical_yn(l, x, derivative=True)
            h_x, dh_x = j_x + 1j * y_x, dj_x + 1j * dy_x
            j_i, dj_i = spherical_jn(l, xi), spherical_jn(l, xi, derivative=True)
            Dj_x, Dh_x, Dj_i = _d_xz(j_x, x, dj_x), _d_xz(h_x, x, dh_x), _d_xz(j_i, xi, dj_i)
            Q[i, 0, l - 1] = (j_x * Dj_i - j_i * Dj_x) / (j_i * Dh_x - h_x * Dj_i)                       # (B.2)
            Q[i, 1, l - 1] = (k**2 * j_x * Dj_i - ki**2 * j_i * Dj_x) / (ki**2 * j_i * Dh_x - k**2 * h_x * Dj_i)  # (B.3)
    return Q


def t_diagonal(q, lmax) -> np.ndarray:
    """Diagonal of T^i (B.1): T_n = Q_{tau,l}, independent of m.  [N, nmax]."""
    q = np.asarray(q)
    idx = multi_indices(lmax)
    return np.stack([q[:, tau - 1, l - 1] for (tau, l, m) in idx], axis=1)


def system_matvec(pos, k, lmax, q, b) -> np.ndarray:
    """sum_{i',n'} M^{ii'}_{nn'} b^{i'}_{n'} = b - T (W b), eqs. (8)-(9)."""
    N = np.asarray(pos).shape[0]
    b = np.asarray(b, dtype=np.complex128).reshape(N, nmax_of(lmax))
    return b - t_diagonal(q, lmax) * coupling_matvec(pos, k, lmax, b)


def rhs(q, lmax, a_in) -> np.ndarray:
    """Right-hand side of eq. (8): T a_in."""
    return t_diagonal(q, lmax) * np.asarray(a_in, dtype=np.complex128)


# ----------------------------------------------------------------------------- angular functions
def legendre_pi_tau(lmax, ct, st):
    """Normalised P_l^m, pi_l^m = P_l^m / sin(theta), tau_l^m = d/dtheta P_l^m (A.3),
    0 <= m <= l <= lmax, by the three-term recursion of reading R2 (no Condon-Shortley phase).
    ct, st: arrays of cos(theta), sin(theta).  Returns three dicts keyed (l, m) of arrays.
    pi_l^0 is returned as 0: it only ever appears multiplied by m = 0."""
    ct = np.asarray(ct, dtype=np.float64); st = np.asarray(st, dtype=np.float64)
    P, pi, tau = {}, {}, {}
    P[(0, 0)] = np.full_like(ct, 1.0 / np.sqrt(2.0))
    for mu in range(0, lmax + 1):
        if mu > 0:
            c = np.sqrt((2 * mu + 1) / (2 * mu))
            P[(mu, mu)] = c * st * P[(mu - 1, mu - 1)]
            pi[(mu, mu)] = c * P[(mu - 1, mu - 1)]
        else:
            pi[(0, 0)] = np.zeros_like(ct)
        if mu + 1 <= lmax:
            P[(mu + 1, mu)] = np.sqrt(2 * mu + 3) * ct * P[(mu, mu)]
            pi[(mu + 1, mu)] = np.sqrt(2 * mu + 3) * ct * pi[(mu, mu)]
        for p in range(mu + 2, lmax + 1):
            f1 = np.sqrt((4 * p * p - 1) / (p * p - mu * mu))
            f2 = np.sqrt(((p - 1) ** 2 - mu * mu) / (4 * (p - 1) ** 2 - 1))
            P[(p, mu)] = f1 * (ct * P[(p - 1, mu)] - f2 * P[(p - 2, mu)])
            pi[(p, mu)] = f1 * (ct * pi[(p - 1, mu)] - f2 * pi[(p - 2, mu)])
    for l in range(0, lmax + 1):
        for m in range(0, l + 1):
            if m == 0:
                # d/dtheta P_l^0 = -sqrt(l(l+1)) P_l^1
                tau[(l, 0)] = -np.sqrt(l * (l + 1)) * P[(l, 1)] if l >= 1 else np.zeros_like(ct)
            else:
                # sin(theta) dP/dtheta = l cos(theta) P_l^m - (l+m) (N_lm/N_{l-1,m}) P_{l-1}^m
                prev = pi[(l - 1, m)] if (l - 1) >= m else np.zeros_like(ct)
                ratio = np.sqrt((2 * l + 1) / (2 * l - 1) * (l - m) / (l + m))
                tau[(l, m)] = l * ct * pi[(l, m)] - (l + m) * ratio * prev
    return P, pi, tau


# ----------------------------------------------------------------------------- SVWFs (A.2), PVWFs (A.4)
def _radial_np(nu, l, x):
    if nu == 1:
        return spherical_jn(l, x) + 0j, spherical_jn(l, x, derivative=True) + 0j
    return (spherical_jn(l, x) + 1j * spherical_yn(l, x),
            spherical_jn(l, x, derivative=True) + 1j * spherical_yn(l, x, derivative=True))


def svwf(nu, tau, l, m, k, r) -> np.ndarray:
    """Psi^{(nu)}_{tau l m}(r), explicit form (A.2).  r: [npts,3] Cartesian.
    Returns [npts,3] complex Cartesian components."""
    r = np.atleast_2d(np.asarray(r, dtype=np.float64))
    x, y, z = r[:, 0], r[:, 1], r[:, 2]
    rr = np.sqrt(x * x + y * y + z * z)
    rho = np.sqrt(x * x + y * y)
    ct, st = z / rr, rho / rr
    phi = np.arctan2(y, x)
    cp, sp = np.cos(phi), np.sin(phi)
    e_r = np.stack([st * cp, st * sp, ct], axis=1)
    e_t = np.stack([ct * cp, ct * sp, -st], axis=1)
    e_p = np.stack([-sp, cp, np.zeros_like(sp)], axis=1)
    P, pi, tau_ = legendre_pi_tau(l, ct, st)
    am = abs(m)
    Plm, pilm, taulm = P[(l, am)], pi[(l, am)], tau_[(l, am)]
    kr = k * rr
    zl, dzl = _radial_np(nu, l, kr)
    pref = np.exp(1j * m * phi) / np.sqrt(2.0 * l * (l + 1))
    if tau == 1:
        F = (pref * zl)[:, None] * ((1j * m * pilm)[:, None] * e_t - taulm[:, None] * e_p)
    else:
        dxz = (zl + kr * dzl) / kr                  # d_{kr}(kr z_l(kr)) / kr
        F = pref[:, None] * ((l * (l + 1) * zl / kr * Plm)[:, None] * e_r
                             + dxz[:, None] * (taulm[:, None] * e_t + (1j * m * pilm)[:, None] * e_p))
    return F


def pvwf(j, alpha, beta, k, r) -> np.ndarray:
    """Phi_j(alpha, beta; r) = exp(i k.r) e_alpha (j=1) or e_beta (j=2), (A.4)."""
    r = np.atleast_2d(np.asarray(r, dtype=np.float64))
    kvec = k * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
    e_alpha = np.array([-np.sin(alpha), np.cos(alpha), 0.0])
    e_beta = np.array([np.cos(beta) * np.cos(alpha), np.cos(beta) * np.sin(alpha), -np.sin(beta)])
    e = e_alpha if j == 1 else e_beta
    return np.exp(1j * (r @ kvec))[:, None] * e[None, :]


def plane_wave_B(lmax, beta, j, dagger=False) -> np.ndarray:
    """B_{nj}(beta) of (A.14); dagger=True sets every explicit i to -i."""
    ct, st = np.array([np.cos(beta)]), np.array([np.sin(beta)])
    _, pi, tau_ = legendre_pi_tau(lmax, ct, st)
    I = -1j if dagger else 1j
    out = np.zeros(nmax_of(lmax), dtype=np.complex128)
    for (tau, l, m) in multi_indices(lmax):
        am = abs(m)
        ang = tau_[(l, am)][0] if tau == j else m * pi[(l, am)][0]
        pol = I if j == 1 else 1.0
        out[nindex(lmax, tau, l, m)] = -1.0 / (I ** (l + 1)) / np.sqrt(2.0 * l * (l + 1)) * pol * ang
    return out


def plane_wave_a_in(pos, k, lmax, alpha=0.0, beta=0.0, j=2, E0=1.0) -> np.ndarray:
    """Initial-field coefficients of a plane wave E0 Phi_j(alpha, beta; r) about every sphere centre:
    (A.13) gives Phi_j(r) = 4 sum_n e^{-i m alpha} B^dagger_{nj}(beta) Psi^(1)_n(r); shifting the origin to
    r_i multiplies by exp(i k.r_i).  beta = 0, alpha = 0, j = 2 is +z propagation, x-polarised.  [N,nmax]."""
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    kvec = k * np.array([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)])
    Bd = plane_wave_B(lmax, beta, j, dagger=True)
    ms = np.array([m for (_, _, m) in multi_indices(lmax)])
    coeff = 4.0 * np.exp(-1j * ms * alpha) * Bd
    return E0 * np.exp(1j * (pos @ kvec))[:, None] * coeff[None, :]


# ----------------------------------------------------------------------------- reference solves of eq. (8)
def dense_coupling_matrix(pos, k, lmax, kind=3) -> np.ndarray:
    """Full W, [N*nmax, N*nmax], zero diagonal blocks (sum over i' != i)."""
    pos = np.asarray(pos, dtype=np.float64)
    N, n = pos.shape[0], nmax_of(lmax)
    W = np.zeros((N * n, N * n), dtype=np.complex128)
    for i in range(N):
        for ip in range(N):
            if i != ip:
                W[i * n:(i + 1) * n, ip * n:(ip + 1) * n] = coupling_block(lmax, k, pos[i] - pos[ip], kind)
    return W


def dense_system_matrix(pos, k, lmax, q) -> np.ndarray:
    """M = 1 - T W, eq. (9)."""
    N, n = np.asarray(pos).shape[0], nmax_of(lmax)
    T = t_diagonal(q, lmax).reshape(N * n)
    return np.eye(N * n, dtype=np.complex128) - T[:, None] * dense_coupling_matrix(pos, k, lmax)


def solve_dense(pos, k, lmax, q, a_in) -> np.ndarray:
    """b solving eq. (8) by dense LU (numpy.linalg.solve).  Small N only."""
    N, n = np.asarray(pos).shape[0], nmax_of(lmax)
    M = dense_system_matrix(pos, k, lmax, q)
    return np.linalg.solve(M, rhs(q, lmax, a_in).reshape(N * n)).reshape(N, n)


# ----------------------------------------------------------------------------- block-diagonal preconditioner
def cuboid_partition(pos, edge_xyz):
    """Step 1 of PAPER.md:111: divide the volume occupied by the spheres into an array of cuboids (edge lengths
    edge_xyz, anchored at the minimum corner of the centres; an edge <= 0 means no cut along that axis).  Returns a
    list of index arrays, one per non-empty cuboid, cuboids in lexicographic (cx, cy, cz) order, spheres in
    index order inside a cuboid."""
    pos = np.asarray(pos, dtype=np.float64)
    e = np.broadcast_to(np.asarray(edge_xyz, dtype=np.float64), (3,))
    cells = np.zeros(pos.shape, dtype=np.int64)
    for a in range(3):
        if e[a] > 0:
            cells[:, a] = np.floor((pos[:, a] - pos[:, a].min()) / e[a]).astype(np.int64)
    groups = {}
    for i in range(pos.shape[0]):
        groups.setdefault(tuple(cells[i]), []).append(i)
    return [np.array(groups[key], dtype=np.int64) for key in sorted(groups)]


def precond_apply(pos, k, lmax, q, edge_xyz, v) -> np.ndarray:
    """Steps 2-4 of PAPER.md:112-114: z = blockdiag(M_j^{-1}) v with M_j = M restricted to the spheres of G_j,
    each block solved by dense LU (numpy.linalg.solve)."""
    pos = np.asarray(pos, dtype=np.float64)
    N, n = pos.shape[0], nmax_of(lmax)
    v = np.asarray(v, dtype=np.complex128).reshape(N, n)
    z = np.zeros_like(v)
    for idx in cuboid_partition(pos, edge_xyz):
        Mj = dense_system_matrix(pos[idx], k, lmax, np.asarray(q)[idx])
        z[idx] = np.linalg.solve(Mj, v[idx].reshape(-1)).reshape(len(idx), n)
    return z


def solve_gmres(pos, k, lmax, q, a_in, rtol=1e-10, restart=200, max_matvecs=2000, x0=None):
    """b solving eq. (8) by restarted GMRES (Saad & Schultz; ref. [26] of the paper) in FP64 with modified
    Gram-Schmidt; the small least-squares problem is solved with numpy.linalg.lstsq at every step (plain, not
    Givens).  Stops when ||rhs - M x|| / ||rhs|| <= rtol.  Returns (b [N,nmax], info dict)."""
    N, n = np.asarray(pos).shape[0], nmax_of(lmax)
    f = rhs(q, lmax, a_in).reshape(N * n)
    A = lambda v: system_matvec(pos, k, lmax, q, v.reshape(N, n)).reshape(N * n)
    x = np.zeros_like(f) if x0 is None else np.asarray(x0, dtype=np.complex128).reshape(N * n).copy()
    fn = np.linalg.norm(f)
    matvecs, hist = 0, []
    while True:
        r = f - A(x); matvecs += 1
        beta = np.linalg.norm(r)
        hist.append(beta / fn)
        if beta / fn <= rtol or matvecs >= max_matvecs:
            break
        V = [r / beta]
        H = np.zeros((restart + 1, restart), dtype=np.complex128)
        yk = None
        for jj in range(restart):
            w = A(V[jj]); matvecs += 1
            for ii in range(jj + 1):
                H[ii, jj] = np.vdot(V[ii], w)
                w = w - H[ii, jj] * V[ii]
            H[jj + 1, jj] = np.linalg.norm(w)
            e1 = np.zeros(jj + 2, dtype=np.complex128); e1[0] = beta
            yk, *_ = np.linalg.lstsq(H[:jj + 2, :jj + 1], e1, rcond=None)
            res = np.linalg.norm(e1 - H[:jj + 2, :jj + 1] @ yk) / fn
            hist.append(res)
            if res <= rtol or H[jj + 1, jj] == 0 or matvecs >= max_matvecs:
                break
            V.append(w / H[jj + 1, jj])
        x = x + sum(yk[ii] * V[ii] for ii in range(len(yk)))
    return x.reshape(N, n), {"matvecs": matvecs, "rel_residual": hist[-1], "history": hist}


# ----------------------------------------------------------------------------- cross sections (pins P5, P8)
def extinction_cross_section(k, a_in, b) -> float:
    """C_ext = -(pi/k^2) Re sum_{i,n} conj(a_in) b for a unit-amplitude plane wave (optical theorem in the
    SVWF normalisation of A.1-A.2; pinned against the Mie series in tests, P5)."""
    return float(-(np.pi / k**2) * np.real(np.vdot(np.asarray(a_in), np.asarray(b))))


def scattering_cross_section(pos, k, lmax, b) -> float:
    """C_sca = (pi/k^2) Re[ b^H (b + R b) ], R = coupling operator with j_p in place of h_p^(1)
    (the regular translation operator re-expands every sphere's outgoing field about a common origin)."""
    b = np.asarray(b, dtype=np.complex128)
    Rb = coupling_matvec(pos, k, lmax, b, kind=1) if b.shape[0] > 1 else np.zeros_like(b)
    return float((np.pi / k**2) * np.real(np.vdot(b, b + Rb)))


# ----------------------------------------------------------------------------- far field (A.12, D.1-D.3)
def far_field_amplitude(pos, k, lmax, b, alpha, beta) -> np.ndarray:
    """Plane-wave amplitudes g_j(alpha, beta), j = 1, 2, of the scattered field (3) in the directions (alpha, beta)
    (real polar angle beta: the propagating part of D.1).  Each sphere's outgoing SVWFs are turned into
    plane waves with (A.12), about its own centre; shifting the origin to r_i multiplies
    Phi_j(alpha, beta; r - r_i) by exp(-i k.r_i); the contributions of all spheres are added:

        g_j(alpha, beta) = (1 / 2 pi) sum_i exp(-i k(alpha,beta).r_i) sum_n b^i_n B_nj(beta) exp(i m alpha).

    Returns [n_dir, 2] complex128.  The radiant intensity is I_j = 2 pi^2 / (omega k mu_0) |g_j|^2 (D.3)."""
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    b = np.asarray(b, dtype=np.complex128).reshape(pos.shape[0], nmax_of(lmax))
    alpha = np.atleast_1d(np.asarray(alpha, dtype=np.float64))
    beta = np.atleast_1d(np.asarray(beta, dtype=np.float64))
    ms = np.array([m for (_, _, m) in multi_indices(lmax)])
    g = np.zeros((alpha.shape[0], 2), dtype=np.complex128)
    for d in range(alpha.shape[0]):
        kvec = k * np.array([np.sin(beta[d]) * np.cos(alpha[d]), np.sin(beta[d]) * np.sin(alpha[d]), np.cos(beta[d])])
        phase = np.exp(-1j * (pos @ kvec))
        for j in (1, 2):
            c = plane_wave_B(lmax, beta[d], j) * np.exp(1j * ms * alpha[d])
            g[d, j - 1] = np.sum(phase * (b @ c)) / (2.0 * np.pi)
    return g


def scattered_power_cross_section(k, g, weights) -> float:
    """(D.2) as a cross section for a unit-amplitude incident plane wave: the flux P = 2 pi^2 / (omega k mu_0)
    sum_j int |g_j|^2 sin(beta) d(beta) d(alpha) divided by the incident intensity k / (2 omega mu_0) gives
    (4 pi^2 / k^2) sum_j int |g_j|^2 dOmega; `weights` are the quadrature weights of the directions (dOmega)."""
    return float(4.0 * np.pi**2 / k**2 * np.sum(np.asarray(weights)[:, None] * np.abs(g) ** 2))


# ----------------------------------------------------------------------------- Gaussian beam (Appendix C, D.4-D.5)
def _beam_polarisation(j, alpha, alpha_G):
    """(C.3)-(C.4): e^{i(a-aG)} (d_j1 - i d_j2)/2 + e^{-i(a-aG)} (d_j1 + i d_j2)/2."""
    d1, d2 = (1.0, 0.0) if j == 1 else (0.0, 1.0)
    return np.exp(1j * (alpha - alpha_G)) * (d1 - 1j * d2) / 2 + np.exp(-1j * (alpha - alpha_G)) * (d1 + 1j * d2) / 2


def gaussian_beam_a_in(pos, k, lmax, w, r_G, alpha_G=0.0, E0=1.0, n_beta=400) -> np.ndarray:
    """Initial-field coefficients of the Gaussian beam of Appendix C (waist w at r_G, propagating along +z,
    polarisation angle alpha_G), (C.8), with the alpha-integral I_jn(beta) of (C.7)
    (readings R20: I_j of C.8 is I_jn, B_jn^dagger of C.6 is B_nj^dagger).  The beta-integral over [0, pi/2] is
    evaluated with n_beta Gauss-Legendre nodes.  Returns [N, nmax] complex128."""
    from scipy.special import jv
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    rel = pos - np.asarray(r_G, dtype=np.float64)[None, :]
    rho, phi, z = np.hypot(rel[:, 0], rel[:, 1]), np.arctan2(rel[:, 1], rel[:, 0]), rel[:, 2]
    x, wq = np.polynomial.legendre.leggauss(n_beta)
    beta, wq = (x + 1.0) * np.pi / 4.0, wq * np.pi / 4.0
    idx = multi_indices(lmax)
    a = np.zeros((pos.shape[0], nmax_of(lmax)), dtype=np.complex128)
    for q in range(n_beta):
        sb, cb = np.sin(beta[q]), np.cos(beta[q])
        common = wq[q] * sb * cb * np.exp(-w * w * k * k * sb * sb / 4.0) * np.exp(1j * k * z * cb)      # [N]
        for j in (1, 2):
            Bd = plane_wave_B(lmax, beta[q], j, dagger=True)
            d1, d2 = (1.0, 0.0) if j == 1 else (0.0, 1.0)
            for n, (tau, l, m) in enumerate(idx):
                I = (2 * np.pi * np.exp(-1j * alpha_G) * 1j ** abs(m - 1) * np.exp(-1j * (m - 1) * phi)
                     * jv(abs(m - 1), k * rho * sb) * (d1 - 1j * d2) / 2
                     + 2 * np.pi * np.exp(1j * alpha_G) * 1j ** abs(m + 1) * np.exp(-1j * (m + 1) * phi)
                     * jv(abs(m + 1), k * rho * sb) * (d1 + 1j * d2) / 2)
                a[:, n] += common * Bd[n] * I
    return E0 * k * k * w * w / np.pi * a


def gaussian_beam_a_in_brute_force(pos, k, lmax, w, r_G, alpha_G=0.0, E0=1.0, n_beta=200, n_alpha=256) -> np.ndarray:
    """The same coefficients straight from the angular spectrum (C.4), with the exact phase
    e^{i k.(r_i - r_G)} (the product of the two exponentials of (C.5), reading R20) and (A.13) for every plane wave;
    both integrals by quadrature (uniform in alpha, Gauss-Legendre in beta).  Small N only."""
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    rel = pos - np.asarray(r_G, dtype=np.float64)[None, :]
    x, wq = np.polynomial.legendre.leggauss(n_beta)
    beta, wq = (x + 1.0) * np.pi / 4.0, wq * np.pi / 4.0
    alpha = 2 * np.pi * np.arange(n_alpha) / n_alpha
    ms = np.array([m for (_, _, m) in multi_indices(lmax)])
    a = np.zeros((pos.shape[0], nmax_of(lmax)), dtype=np.complex128)
    for q in range(n_beta):
        sb, cb = np.sin(beta[q]), np.cos(beta[q])
        amp = wq[q] * sb * cb * np.exp(-w * w * k * k * sb * sb / 4.0) * (2 * np.pi / n_alpha)
        kvec = k * np.stack([sb * np.cos(alpha), sb * np.sin(alpha), np.full_like(alpha, cb)], axis=1)      # [na, 3]
        phase = np.exp(1j * (rel @ kvec.T))                                                                 # [N, na]
        for j in (1, 2):
            Bd = plane_wave_B(lmax, beta[q], j, dagger=True)
            pol = _beam_polarisation(j, alpha, alpha_G)                                                     # [na]
            # Phi_j(alpha, beta; r - r_i) = 4 sum_n e^{-i m alpha} B^dagger_nj Psi_n^(1)(r - r_i)   (A.13)
            a += amp * (phase * pol[None, :]) @ (4.0 * np.exp(-1j * np.outer(alpha, ms)) * Bd[None, :])
    return E0 * k * k * w * w / (4 * np.pi) * a


def gaussian_beam_g(k, w, r_G, alpha, beta, alpha_G=0.0, E0=1.0) -> np.ndarray:
    """Plane-wave amplitudes of the beam, (D.4), for polarisation angle alpha_G (D.4 prints alpha_G = 0):
    g_j = E0 k^2 w^2 / (4 pi) cos(beta) exp(-w^2 k^2 sin^2(beta) / 4) (d_j1 cos(a - aG) + d_j2 sin(a - aG)) e^{-i k.r_G};
    zero for beta > pi/2 (the beam only contains waves travelling towards +z).  [n_dir, 2]."""
    alpha = np.atleast_1d(np.asarray(alpha, dtype=np.float64)); beta = np.atleast_1d(np.asarray(beta, dtype=np.float64))
    kvec = k * np.stack([np.sin(beta) * np.cos(alpha), np.sin(beta) * np.sin(alpha), np.cos(beta)], axis=1)
    amp = E0 * k * k * w * w / (4 * np.pi) * np.cos(beta) * np.exp(-w * w * k * k * np.sin(beta) ** 2 / 4.0)
    amp = np.where(beta <= np.pi / 2, amp, 0.0) * np.exp(-1j * (kvec @ np.asarray(r_G, dtype=np.float64)))
    return np.stack([amp * np.cos(alpha - alpha_G), amp * np.sin(alpha - alpha_G)], axis=1)


# ----------------------------------------------------------------------------- near field (eq. 3)
def scattered_field(pos, k, lmax, b, points) -> np.ndarray:
    """E_scat(r) = sum_i sum_n b^i_n Psi^(3)_n(r - r_i), eq. (3), with svwf() ((A.2); pinned by P1, P2).
    points [n_pts, 3] outside every sphere.  Returns [n_pts, 3] complex128 Cartesian components."""
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    pts = np.atleast_2d(np.asarray(points, dtype=np.float64))
    b = np.asarray(b, dtype=np.complex128).reshape(pos.shape[0], nmax_of(lmax))
    E = np.zeros((pts.shape[0], 3), dtype=np.complex128)
    idx = multi_indices(lmax)
    for i in range(pos.shape[0]):
        rel = pts - pos[i][None, :]
        for n, (tau, l, m) in enumerate(idx):
            E += b[i, n] * svwf(3, tau, l, m, k, rel)
    return E
