"""The boundary is a C ABI: include/celes.h must be plain C, and a C99 program with no CUDA or Python in it must be
able to drive the library through the host-buffer entry points."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_abi", "c_abi_smoke.c")
INC = os.path.join(ROOT, "include")
PKG = os.path.join(ROOT, "paper_1706_02145_b200")


def test_header_and_client_are_plain_c99():
    """gcc -std=c99 -pedantic-errors -Wall -Werror parses the header through the C client (no GPU, no link)."""
    r = subprocess.run(["gcc", "-std=c99", "-pedantic-errors", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-I", INC, SRC],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_c_client_links_against_the_library(tmp_path):
    """Link step only (no GPU needed): every symbol the C client uses is exported with C linkage."""
    from paper_1706_02145_b200 import build
    build.build()
    exe = tmp_path / "c_abi_smoke"
    r = subprocess.run(["gcc", "-std=c99", "-O1", "-I", INC, SRC, "-o", str(exe), "-L", PKG, "-lceles",
                        f"-Wl,-rpath,{PKG}"], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    # without a GPU (or with a bad file) the program must fail cleanly, not crash
    r = subprocess.run([str(exe), str(tmp_path / "missing.bin"), str(tmp_path / "out.bin")], capture_output=True, text=True)
    assert r.returncode == 2


@pytest.mark.gpu
def test_c_client_matches_oracle(tmp_path):
    sys.path.insert(0, ROOT)
    from oracle import celes_oracle as orc
    from paper_1706_02145_b200 import build, fields, workloads
    build.build()
    exe = tmp_path / "c_abi_smoke"
    subprocess.run(["gcc", "-std=c99", "-O1", "-I", INC, SRC, "-o", str(exe), "-L", PKG, "-lceles", f"-Wl,-rpath,{PKG}"],
                   check=True)
    w = workloads.C1
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    b = workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)
    with open(tmp_path / "in.bin", "wb") as f:
        f.write(np.array([w.N, w.lmax], dtype=np.int32).tobytes())
        f.write(np.array([w.k], dtype=np.float64).tobytes())
        f.write(np.ascontiguousarray(pos, dtype=np.float64).tobytes())
        f.write(np.ascontiguousarray(rad, dtype=np.float64).tobytes())
        f.write(np.ascontiguousarray(q, dtype=np.complex128).tobytes())
        f.write(np.ascontiguousarray(b, dtype=np.complex64).tobytes())
    r = subprocess.run([str(exe), str(tmp_path / "in.bin"), str(tmp_path / "out.bin")], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    res = np.fromfile(tmp_path / "out.bin", dtype=np.complex64).reshape(2, w.N, w.nmax)
    ref = orc.coupling_matvec(pos, w.k, w.lmax, b)
    qo = orc.mie_q(w.lmax, w.k, rad, workloads.N_SPHERE)
    rel = lambda a, c: np.linalg.norm(a - c) / np.linalg.norm(c)
    assert rel(res[0], ref) <= 1e-4
    assert rel(res[1], orc.system_matvec(pos, w.k, w.lmax, qo, b)) <= 1e-4
