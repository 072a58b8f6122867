"""Build step of the CUDA library: nvcc -> paper_1706_02145_b200/libceles.so (in-tree, sm_100a only).

    python -m paper_1706_02145_b200.build [--force] [--regen]

``--regen`` first re-runs both generators of the straight-line pair bodies, csrc/gen_coupling_body.py (direct sum,
lmax 1-4) and csrc/gen_packed_body.py (packed rotated body, lmax 1-5); needs SymPy, the generated files are committed.
nvcc cross-compiles without a GPU.  Five translation units (csrc/celes.cu, solve.cu, precond.cu, fields.cu, probe.cu).  The library is loaded by ``paper_1706_02145_b200.binding`` via ctypes.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libceles.so")
NVCC_FLAGS = ["-std=c++17", "-O3", *os.environ.get("CELES_NVCC_EXTRA", "").split(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC"]
NVCC_LIBS: list[str] = []       # the CUDA runtime only


def sources() -> list[str]:
    out = [os.path.join(HERE, "..", "include", "celes.h")]
    for root, _, files in os.walk(CSRC):
        out += [os.path.join(root, f) for f in files if f.endswith((".cu", ".cuh", ".h", ".inc"))]
    return out


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build(force: bool = False, regen: bool = False, verbose: bool = False) -> str:
    if regen:
        subprocess.run([sys.executable, os.path.join(CSRC, "gen_coupling_body.py")], check=True)
        subprocess.run([sys.executable, os.path.join(CSRC, "gen_packed_body.py")], check=True)
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        units = [os.path.join(CSRC, f) for f in ("celes.cu", "solve.cu", "precond.cu", "fields.cu", "probe.cu")]
        cmd = [nvcc, *NVCC_FLAGS, "--threads", "5", *(["-Xptxas", "-v"] if verbose else []), "-o", LIB, *units, *NVCC_LIBS]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, regen="--regen" in sys.argv, verbose="-v" in sys.argv))
