"""CELES oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain FP64 CPU implementation of the hot path of arxiv 1706.02145, written
from the paper's equations.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import it; the CUDA
path under ``paper_1706_02145_b200/`` never does, and this package never imports that
one.  See ``celes_oracle.cpp`` (coupling operator, eqs. 6-7, A.6-A.11) and
``celes_oracle.py`` (T-matrix B.1-B.3, plane wave A.13-A.14, SVWFs A.2, solve of eq. 8).
"""
from .celes_oracle import *  # noqa: F401,F403
