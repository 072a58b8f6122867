"""The generated pair bodies, compiled for the HOST, against the FP64 oracle (no GPU needed).

tests/host_emulation/pair_body_host.cpp compiles csrc/pair_math.cuh and csrc/generated/*.inc with g++ (the packed
intrinsics emulated with fmaf) and applies one pair's W block in the kernel's work basis.  Here the block is rebuilt
column by column, taken back to the (tau, l, m) basis with the transform that pack_kernel / finalize_kernel document
(csrc/coupling_kernel.cuh), and compared with the oracle's term-by-term (A.6)-(A.11) block.
A wrong sign, index or coefficient anywhere in a generator fails this within seconds, before any GPU run.
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest

from oracle import celes_oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
K = 0.011423973285781066          # 2 pi / 550 nm
F32P = ctypes.POINTER(ctypes.c_float)


@pytest.fixture(scope="module")
def host_lib(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("hostbody") / "libpair_host.so")
    subprocess.run(["g++", "-std=c++17", "-O0", "-shared", "-fPIC", "-I/usr/local/cuda/include",
                    "-I" + os.path.join(ROOT, "paper_1706_02145_b200", "csrc"), "-o", out,
                    os.path.join(ROOT, "tests", "host_emulation", "pair_body_host.cpp")], check=True)
    lib = ctypes.CDLL(out)
    lib.celes_host_pair_body.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, ctypes.c_float, F32P, F32P]
    return lib


def work_basis(lmax, variant):
    """T with b_work = T b: variant 1 (direct) [b_1 + b_2 | b_1 - b_2]; variant 0 (packed rotated) the orthonormal
    [tau S|A][l][u_0, u+_1, w_1, ...] basis, u+-_m = (x_m +- x_-m)/sqrt2, x_S/A = (x_1 +- x_2)/sqrt2, w_m = i u-_m."""
    H = lmax * (lmax + 2)
    T = np.zeros((2 * H, 2 * H), complex)
    if variant == 1:
        for q in range(H):
            T[q, q] = T[q, H + q] = T[H + q, q] = 1.0
            T[H + q, H + q] = -1.0
        return T
    for l in range(1, lmax + 1):
        c0, base = (l - 1) * (l + 1) + l, l * l - 1
        for ts, s2 in ((0, 1.0), (1, -1.0)):
            T[ts * H + base, c0] = np.sqrt(0.5)
            T[ts * H + base, H + c0] = s2 * np.sqrt(0.5)
            for m in range(1, l + 1):
                for pos, sg, ph in ((2 * m - 1, 0.5, 1.0), (2 * m, -0.5, 1j)):
                    row = ts * H + base + pos
                    T[row, c0 + m], T[row, c0 - m] = 0.5 * ph, sg * ph
                    T[row, H + c0 + m], T[row, H + c0 - m] = 0.5 * ph * s2, sg * ph * s2
    return T


def host_block(lib, lmax, variant, kd):
    n = 2 * lmax * (lmax + 2)
    W = np.zeros((n, n), complex)
    for q in range(n):
        b = np.zeros(2 * n, np.float32)
        b[2 * q] = 1.0
        y = np.zeros(2 * n, np.float32)
        assert lib.celes_host_pair_body(lmax, variant, float(kd[0]), float(kd[1]), float(kd[2]),
                                        b.ctypes.data_as(F32P), y.ctypes.data_as(F32P)) == 0
        W[:, q] = y[0::2] + 1j * y[1::2]
    return W


def displacements():
    rng = np.random.default_rng(7)
    ds = [np.array([230.0, 40.0, -60.0]), np.array([0.0, 0.0, 201.0]), np.array([0.0, 0.0, -350.0]),
          np.array([1e-9, 0.0, 400.0]), np.array([201.0, 0.0, 0.0]), np.array([3000.0, -5000.0, 120.0])]
    for s in (150.0, 400.0, 3000.0):
        for _ in range(3):
            d = rng.normal(size=3) * s
            ds.append(d if np.linalg.norm(d) >= 201.0 else d / np.linalg.norm(d) * 201.0)
    return ds


@pytest.mark.parametrize("lmax,variant", [(1, 0), (2, 0), (3, 0), (4, 0), (5, 0), (1, 1), (2, 1), (3, 1), (4, 1)])
def test_generated_pair_body_matches_oracle_block(host_lib, lmax, variant):
    T = work_basis(lmax, variant)
    Tinv = np.linalg.inv(T)
    for d in displacements():
        ref = orc.coupling_block(lmax, K, d)
        kd = (K * d).astype(np.float32)                     # the kernel rounds k (r_i - r_i') once, after the FP64 subtraction
        W = Tinv @ host_block(host_lib, lmax, variant, kd) @ T
        scale = np.abs(ref).max()
        assert np.linalg.norm(W - ref) <= 1e-5 * np.linalg.norm(ref), (lmax, variant, d)
        assert np.abs(W - ref).max() <= 2e-5 * scale, (lmax, variant, d)


def test_host_body_accumulates_into_y(host_lib):
    """y += W b: the body adds to what the accumulator holds (the chains are seeded from it)."""
    lmax, n = 3, 30
    rng = np.random.default_rng(11)
    b = rng.normal(size=2 * n).astype(np.float32)
    y0 = rng.normal(size=2 * n).astype(np.float32)
    kd = (K * np.array([120.0, -260.0, 90.0])).astype(np.float32)
    y = y0.copy()
    z = np.zeros(2 * n, np.float32)
    for buf in (y, z):
        host_lib.celes_host_pair_body(lmax, 0, float(kd[0]), float(kd[1]), float(kd[2]), b.ctypes.data_as(F32P),
                                      buf.ctypes.data_as(F32P))
    assert np.allclose(y - y0, z, rtol=0, atol=2e-5 * np.abs(z).max())
