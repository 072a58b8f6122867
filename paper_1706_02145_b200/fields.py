"""Host-side input preparation for celes_setup / celes_solve: the sphere T-matrix entries and the plane-wave
initial-field coefficients.  O(N) work done once per simulation in FP64 ("multiplication with the
T-matrices scales linearly with N"); the results are INPUTS of the C ABI, not part of the hot path.

Written independently of oracle/ (which evaluates (B.2)-(B.3) and (A.13)-(A.14) literally): here the T-matrix is
expressed through the textbook Lorenz-Mie coefficients in Riccati-Bessel form and the plane wave through its
closed form at normal incidence.  tests/test_host_logic.py compares the two.
"""
from __future__ import annotations

import numpy as np
from scipy.special import spherical_jn, spherical_yn


def mie_coefficients(lmax: int, k: float, radii, n_sphere, n0: float = 1.0) -> np.ndarray:
    """Q^i_{tau,l} (B.1-B.3) as [N, 2, lmax] complex128.

    With x = k R, m = n_i / n_0, psi_l(z) = z j_l(z), xi_l(z) = z h_l^(1)(z):
        a_l = (m psi_l(mx) psi_l'(x) - psi_l(x) psi_l'(mx)) / (m psi_l(mx) xi_l'(x) - xi_l(x) psi_l'(mx))   (TM)
        b_l = (psi_l(mx) psi_l'(x) - m psi_l(x) psi_l'(mx)) / (psi_l(mx) xi_l'(x) - m xi_l(x) psi_l'(mx))   (TE)
    and Q_{1,l} = -b_l, Q_{2,l} = -a_l (reading R11)."""
    radii = np.atleast_1d(np.asarray(radii, dtype=np.float64))
    m = np.broadcast_to(np.asarray(n_sphere, dtype=np.complex128) / n0, radii.shape)
    x = k * radii
    mx = m * x
    ls = np.arange(1, lmax + 1)[None, :]
    X, MX, M = x[:, None], mx[:, None], m[:, None]
    jx, djx = spherical_jn(ls, X), spherical_jn(ls, X, derivative=True)
    yx, dyx = spherical_yn(ls, X), spherical_yn(ls, X, derivative=True)
    jm, djm = spherical_jn(ls, MX), spherical_jn(ls, MX, derivative=True)
    psi_x, dpsi_x = X * jx, jx + X * djx
    xi_x, dxi_x = X * (jx + 1j * yx), (jx + 1j * yx) + X * (djx + 1j * dyx)
    psi_m, dpsi_m = MX * jm, jm + MX * djm
    a = (M * psi_m * dpsi_x - psi_x * dpsi_m) / (M * psi_m * dxi_x - xi_x * dpsi_m)
    b = (psi_m * dpsi_x - M * psi_x * dpsi_m) / (psi_m * dxi_x - M * xi_x * dpsi_m)
    return np.stack([-b, -a], axis=1)


def plane_wave_coefficients(pos, k: float, lmax: int, E0: complex = 1.0) -> np.ndarray:
    """a^i_in of a plane wave travelling along +z, polarised along x, amplitude E0, expanded about every sphere
    centre (from (A.13)-(A.14), at beta = 0):
        a^i_{(tau,l,m)} = E0 e^{i k z_i} (-i^{l+1}) sqrt(2l+1) delta_{|m|,1} * (1 if tau = 2 else m).
    Returns [N, nmax] complex128 in the index order n = (tau-1) nmax/2 + (l-1)(l+1) + (m+l)."""
    pos = np.atleast_2d(np.asarray(pos, dtype=np.float64))
    H = lmax * (lmax + 2)
    c = np.zeros(2 * H, dtype=np.complex128)
    for l in range(1, lmax + 1):
        amp = -(1j ** (l + 1)) * np.sqrt(2 * l + 1)
        for m in (-1, 1):
            q = (l - 1) * (l + 1) + (m + l)
            c[q] = amp * m          # tau = 1
            c[H + q] = amp          # tau = 2
    return E0 * np.exp(1j * k * pos[:, 2])[:, None] * c[None, :]
