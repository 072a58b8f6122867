"""CPU-only checks of the product's host side: the C-ABI library loads and exports every symbol of
include/celes.h, argument validation, the run-time translation table against the oracle's a5/b5 and against
the immediates baked into the generated kernel bodies, and the input-preparation helpers against the oracle."""
import ctypes
import os
import re
import sys

import numpy as np
import pytest

import paper_1706_02145_b200 as celes
from paper_1706_02145_b200 import binding, fields, workloads
from paper_1706_02145_b200 import build as celes_build
from oracle import celes_oracle as orc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    celes_build.build()


def test_library_exports_every_declared_symbol():
    declared = set()
    for name in os.listdir(os.path.join(ROOT, "include")):                 # celes.h and celes_probe.h
        hdr = open(os.path.join(ROOT, "include", name)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared |= set(re.findall(r"\b(celes_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_nmax_and_strerror():
    assert [celes.celes_nmax(l) for l in (1, 2, 3, 4, 5)] == [6, 16, 30, 48, 70]
    with pytest.raises(celes.CelesError):
        celes.celes_nmax(0)
    with pytest.raises(celes.CelesError):
        celes.celes_nmax(6)
    for code in (0, -1, -2, -3, -4, -5):
        assert binding.strerror(code) and "unknown" not in binding.strerror(code)
    assert "unknown" in binding.strerror(-99)


def _setup_rc(N, lmax, pos, rad, q, k, out=True):
    L = binding.lib()
    h = ctypes.c_void_p(123)
    rc = L.celes_setup(ctypes.byref(h) if out else None, N, lmax,
                       None if pos is None else pos.ctypes.data, None if rad is None else rad.ctypes.data,
                       None if q is None else q.ctypes.data, k, None, None)
    return rc, h.value


def test_setup_rejects_bad_arguments_before_touching_the_gpu():
    pos = np.array([[0., 0, 0], [300., 0, 0]]); rad = np.array([100., 100.]); q = np.zeros((2, 2, 3), complex)
    k = 0.0114
    assert _setup_rc(2, 3, pos, rad, q, k, out=False)[0] == binding.CELES_EINVAL
    assert _setup_rc(0, 3, pos, rad, q, k) == (binding.CELES_EINVAL, None)
    assert _setup_rc(2, 0, pos, rad, q, k)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 6, pos, rad, q, k)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 3, None, rad, q, k)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 3, pos, None, q, k)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 3, pos, rad, None, k)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 3, pos, rad, q, 0.0)[0] == binding.CELES_EINVAL
    assert _setup_rc(2, 3, pos, rad, q, float("nan"))[0] == binding.CELES_EINVAL
    bad = pos.copy(); bad[1, 1] = np.inf
    assert _setup_rc(2, 3, bad, rad, q, k)[0] == binding.CELES_EINVAL
    close = pos.copy(); close[1, 0] = 199.0           # overlapping spheres (PAPER.md:33 needs disjoint spheres)
    assert _setup_rc(2, 3, close, rad, q, k)[0] == binding.CELES_EINVAL
    badr = rad.copy(); badr[0] = -1.0
    assert _setup_rc(2, 3, pos, badr, q, k)[0] == binding.CELES_EINVAL


def test_overlap_check_finds_a_single_overlap_in_a_large_packing():
    w = workloads.scaled(workloads.C3, 3000)
    pos, rad = workloads.positions(w)
    q = np.zeros((w.N, 2, w.lmax), complex)
    rc, _ = _setup_rc(w.N, w.lmax, pos, rad, q, w.k)
    assert rc in (binding.CELES_OK, binding.CELES_ECUDA)       # valid packing: passes validation (no GPU here -> ECUDA)
    bad = pos.copy(); bad[1717] = bad[42] + np.array([150.0, 0.0, 10.0])
    assert _setup_rc(w.N, w.lmax, bad, rad, q, w.k)[0] == binding.CELES_EINVAL


def test_default_partition_has_the_measured_level_counts():
    """The level counts the documentation states and the profiles measured (profiles/r02n_levels_small_n.md,
    r02i_kernel_c4.md): with 296 resident CTAs the default guided partition makes ten waves of runs at N = 1e5, three at
    N = 1e4 with tiles of 32 (the halving stops at runs of 16 tiles) and five with the tiles of 8 that lmax = 5 uses; an
    explicit level count still overrides the default downwards."""
    res = 296
    assert celes.celes_plan_work(100000, 32, res, 0, 0)["ctas"] == 10 * res
    assert celes.celes_plan_work(10000, 32, res, 0, 0)["ctas"] == 3 * res
    assert celes.celes_plan_work(10000, 8, res, 0, 0)["ctas"] == 5 * res
    assert celes.celes_plan_work(100000, 32, res, 6, 0)["ctas"] == 6 * res
    assert celes.celes_plan_work(10000, 32, res, 1, 0)["ctas"] == res
    p = celes.celes_plan_work(10000, 32, res, 0, 0)
    assert len(p["segments"]) == 965                                   # the partial-sum slots quoted in DESIGN.md section 5.0
    assert len(celes.celes_plan_work(100000, 32, res, 0, 0)["segments"]) == 3740


def test_without_a_gpu_the_product_fails_loudly_and_never_touches_the_oracle():
    """No CPU fallback (the tier's rule): on a box without a CUDA device a valid celes_setup is CELES_ECUDA and returns no
    context, bench.py's own arm exits non-zero saying so, and importing the product (package + bench) imports nothing of
    oracle/.  Skipped where a GPU is present (the GPU tests cover that side)."""
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    w = workloads.C1
    pos, rad = workloads.positions(w)
    rc, handle = _setup_rc(w.N, w.lmax, pos, rad, np.zeros((w.N, 2, w.lmax), complex), w.k)
    assert rc == binding.CELES_ECUDA and not handle
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1", "--warmup", "0"], cwd=ROOT,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
    assert not [l for l in r.stdout.splitlines() if l.startswith("{")]            # and no number is printed
    code = ("import sys; sys.path.insert(0, %r); import paper_1706_02145_b200, bench; "
            "from paper_1706_02145_b200 import binding, fields, workloads, sharding, sass_count; "
            "bad = [m for m in sys.modules if m == 'oracle' or m.startswith('oracle.')]; print('ORACLE', bad)" % ROOT)
    r = subprocess.run([sys.executable, "-c", code], cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-1500:]
    assert "ORACLE []" in r.stdout


def test_compute_entry_points_reject_null():
    L = binding.lib()
    assert L.celes_coupling_matvec(None, None, None, None) == binding.CELES_EINVAL
    assert L.celes_system_matvec(None, None, None, None) == binding.CELES_EINVAL
    assert L.celes_solve(None, None, None, None, None, None) == binding.CELES_EINVAL
    L.celes_destroy(None)


@pytest.mark.parametrize("lmax", [1, 2, 3, 4, 5])
def test_translation_table_matches_oracle_a5_b5(lmax):
    """The library's run-time table (own 3j code) against the oracle's Racah-formula a5/b5, with the index swap
    of eq. (7): W_{(lm),(l'm')} uses a5(l',m'|l,m|p)."""
    a, b = celes.celes_translation_table(lmax)
    for l in range(1, lmax + 1):
        for m in range(-l, l + 1):
            for lp in range(1, lmax + 1):
                for mp in range(-lp, lp + 1):
                    r, c = (l - 1) * (l + 1) + m + l, (lp - 1) * (lp + 1) + mp + lp
                    for p in range(0, 2 * lmax + 1):
                        va, vb = orc.a5(lp, mp, l, m, p), orc.b5(lp, mp, l, m, p)
                        if p < abs(l - lp) or p > l + lp:
                            assert a[r, c, p] == 0 and b[r, c, p] == 0
                            continue
                        assert abs(va.imag) < 1e-13 and abs(vb.real) < 1e-13
                        assert abs(a[r, c, p] - va.real) < 1e-12
                        assert abs(b[r, c, p] - vb.imag) < 1e-12


@pytest.mark.parametrize("lmax", [1, 2, 3, 4])
def test_generated_kernel_bodies_carry_the_table_counts(lmax):
    """The generated straight-line bodies state how many non-zero a5 / b5 terms (p >= |m'-m|) they contain; the
    same count from the library's table."""
    a, b = celes.celes_translation_table(lmax)
    na = nb = 0
    for l in range(1, lmax + 1):
        for m in range(-l, l + 1):
            for lp in range(1, lmax + 1):
                for mp in range(-lp, lp + 1):
                    r, c = (l - 1) * (l + 1) + m + l, (lp - 1) * (lp + 1) + mp + lp
                    for p in range(abs(mp - m), 2 * lmax + 1):
                        na += abs(a[r, c, p]) > 1e-14
                        nb += abs(b[r, c, p]) > 1e-14
    head = open(os.path.join(ROOT, "paper_1706_02145_b200", "csrc", "generated", f"coupling_body_lmax{lmax}.inc")).read(400)
    mt = re.search(r"a5 (\d+), b5 (\d+)", head)
    assert (int(mt.group(1)), int(mt.group(2))) == (na, nb)


def test_mie_coefficients_match_oracle_B2_B3():
    k = 2 * np.pi / 550.0
    R = np.array([100.0, 80.0, 120.0, 95.5])
    for n in (1.52, 1.52 + 0.1j, 2.4):
        assert np.abs(fields.mie_coefficients(4, k, R, n) - orc.mie_q(4, k, R, n)).max() < 1e-13


def test_plane_wave_coefficients_match_oracle_A13():
    k = 2 * np.pi / 550.0
    pos = np.random.default_rng(5).normal(size=(7, 3)) * 400
    for lmax in (1, 3, 4):
        a = fields.plane_wave_coefficients(pos, k, lmax)
        assert np.abs(a - orc.plane_wave_a_in(pos, k, lmax)).max() < 1e-13


def test_workloads_are_seeded_and_valid():
    w = workloads.C1
    p1, r1 = workloads.positions(w)
    p2, _ = workloads.positions(w)
    assert np.array_equal(p1, p2)
    assert workloads.min_gap(p1, r1) >= workloads.GAP_NM - 1e-9
    b = workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)
    assert b.dtype == np.complex64 and b.shape == (50, 30)
    assert abs(np.mean(np.abs(b) ** 2) - 1.0) < 0.1


def test_partition_matches_oracle_cuboids():
    """celes_partition (host side of celes_precond_setup) against the oracle's cuboid partition:
    same subsets, same numbering (lexicographic cuboid order)."""
    w = workloads.scaled(workloads.C3, 1500)
    pos, _ = workloads.positions(w)
    for edge in ([1000.0, 1500.0, 0.0], [800.0, 800.0, 100.0], [0.0, 0.0, 0.0], 2500.0):
        g, n = celes.celes_partition(pos, edge)
        ref = orc.cuboid_partition(pos, edge)
        assert n == len(ref)
        for j, idx in enumerate(ref):
            assert np.all(g[idx] == j)
    with pytest.raises(celes.CelesError):
        celes.celes_partition(np.array([[np.nan, 0.0, 0.0]]), 1.0)


@pytest.mark.parametrize("gen,prefix", [("gen_coupling_body", "coupling_body"), ("gen_packed_body", "coupling_pk")])
def test_committed_generated_bodies_are_what_the_generators_write(gen, prefix, tmp_path):
    """The straight-line pair bodies under csrc/generated/ are build inputs: regenerate lmax = 1, 2 (seconds, SymPy)
    and compare byte for byte with the committed files."""
    csrc = os.path.join(ROOT, "paper_1706_02145_b200", "csrc")
    sys.path.insert(0, csrc)
    try:
        mod = __import__(gen)
        for lmax in (1, 2):
            mod.emit(lmax, outdir=str(tmp_path))
            new = open(tmp_path / f"{prefix}_lmax{lmax}.inc").read()
            old = open(os.path.join(csrc, "generated", f"{prefix}_lmax{lmax}.inc")).read()
            assert new == old
    finally:
        sys.path.remove(csrc)


@pytest.mark.parametrize("N,etile,res,levels,splits", [(1, 32, 296, 0, 0), (50, 32, 296, 0, 0), (1000, 32, 296, 0, 0),
                                                        (10000, 32, 296, 0, 0), (100000, 32, 296, 0, 0), (10000, 24, 444, 3, 0),
                                                        (333, 7, 5, 4, 0), (10000, 32, 296, 1, 0), (100000, 32, 296, 1, 0),
                                                        (10000, 32, 296, 0, 6), (50, 32, 296, 0, 4), (257, 32, 296, 0, 1)])
def test_work_partition_covers_every_pair_once(N, etile, res, levels, splits):
    """csrc/work_partition.h through celes_plan_work: every (receiver block, emitter) is in exactly one segment, runs are
    tile-aligned, the slots of a receiver block are contiguous and ordered by emitter, the runs of one level are equal
    within one tile and every level is about half as long as the one before."""
    p = celes.celes_plan_work(N, etile, res, levels, splits)
    seg, bs = p["segments"], p["receivers_per_block"]
    rblocks = -(-N // bs)
    assert 1 <= bs <= 128 and rblocks * bs >= N and (rblocks - 1) * bs < N
    assert sorted(seg[:, 4]) == list(range(len(seg)))                  # every slot written by exactly one segment
    assert np.all(np.diff(seg[:, 0]) >= 0) and seg[:, 0].max() == p["ctas"] - 1
    for r in range(rblocks):
        mine = seg[seg[:, 1] == r]
        mine = mine[np.argsort(mine[:, 2])]
        assert len(mine) >= 1 and np.all(np.diff(mine[:, 4]) == 1)      # contiguous slots, in emitter order
        assert mine[0, 2] == 0 and mine[-1, 3] == N
        assert np.array_equal(mine[1:, 2], mine[:-1, 3])                # back to back, no gap, no overlap
        assert np.all(mine[:, 2] % etile == 0) and np.all(mine[:, 3] > mine[:, 2])
    tiles = np.zeros(p["ctas"], dtype=np.int64)
    np.add.at(tiles, seg[:, 0], -(-(seg[:, 3] - seg[:, 2]) // etile))
    if splits == 0:
        lv = levels or 10                                               # CELES_DEFAULT_LEVELS
        assert p["ctas"] <= res * lv and len(seg) <= p["ctas"] + rblocks * lv
        assert np.all(np.diff(tiles) <= 1)                              # runs never grow along the launch order
        if levels == 1:
            assert p["ctas"] <= res and tiles.max() - tiles.min() <= 1  # one wave, equal work
        if p["ctas"] > res and tiles[0] >= 64:
            assert 0.4 <= tiles[res] / tiles[0] <= 0.6                  # second level: half the run length
    else:
        assert p["ctas"] == len(seg) and len(seg) <= rblocks * splits


def test_sass_counts_of_the_built_library_match_the_committed_record():
    """The roofline numerators bench.py reports (flops and FMA-pipe lane operations per pair) are the opcode counts of
    the coupling kernel's per-pair loop in the BUILT libceles.so (paper_1706_02145_b200/sass_count.py, cuobjdump; no
    GPU needed).  The committed csrc/generated/sass_counts.json must equal them, so a generator edit that changes the
    kernel cannot leave stale constants behind; and the packed body keeps its op mix."""
    from paper_1706_02145_b200 import sass_count
    if sass_count.cuobjdump() is None:
        pytest.skip("cuobjdump not installed")
    live = sass_count.summary()
    assert live == sass_count.committed(), "run: python -m paper_1706_02145_b200.sass_count --write"
    for key, c in live.items():
        f = c["fp32"]
        assert c["flops_per_pair"] == 4 * f["FFMA2"] + 2 * (f["FMUL2"] + f["FADD2"]) + 2 * f["FFMA"] + f["FMUL"] + f["FADD"]
        assert c["lane_ops_per_pair"] == 2 * (f["FFMA2"] + f["FMUL2"] + f["FADD2"]) + f["FFMA"] + f["FMUL"] + f["FADD"]
    r3 = live["rotated/3"]
    assert r3["packed_non_fma"] < 200 and r3["fp32"]["FADD2"] <= 2
    assert r3["flops_per_pair"] / r3["lane_ops_per_pair"] > 1.75      # nearly every FMA-pipe slot is an FMA
    b = sass_count.counts_for_bench(3)
    assert b["flops_per_pair"] == r3["flops_per_pair"] and "live" in b["source"]
