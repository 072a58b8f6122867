"""Seeded synthetic inputs shared by the tests, bench.py and the oracle checks.

This module holds NONE of the method's arithmetic (no special functions, no translation
coefficients, no T-matrix): only sphere packings by random sequential addition (RSA), radii,
and complex Gaussian coefficient vectors.  It is the one module both the CUDA path's tests and
the oracle's tests may take inputs from (the two implementations share nothing else).

The paper's workloads are dense disordered packings of equal spheres (R = 100 nm, n = 1.5,
lambda = 532 nm, 10 %-50 % volume fraction, 10^4-10^5 spheres).  Its
particle files are not available; the RSA ensembles C1-C5 of BASELINE.json stand in for them
(DESIGN.md section 4 states the recipe and the readings R15-R18 it relies on).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

GAP_NM = 1.0            # minimum surface-to-surface gap (reading R16)
WAVELENGTH_NM = 550.0   # vacuum wavelength of every BASELINE.json config
N_SPHERE = 1.52         # refractive index of the spheres, lossless
N_BACKGROUND = 1.0


@dataclass(frozen=True)
class Workload:
    name: str
    N: int
    lmax: int
    radius_lo: float
    radius_hi: float
    shape: str             # "cube" or "slab"
    lateral_nm: float      # cube edge (if given) or slab lateral size; 0 -> derived from filling fraction
    filling: float         # filling fraction of the box that holds the CENTRES (reading R15); 0 -> box given
    seed_pos: int
    seed_rad: int
    seed_b: int

    @property
    def nmax(self) -> int:
        return 2 * self.lmax * (self.lmax + 2)

    @property
    def k(self) -> float:
        """background wavenumber in 1/nm"""
        return 2.0 * np.pi * N_BACKGROUND / WAVELENGTH_NM


# BASELINE.json configs[0..4]
C1 = Workload("C1", 50, 3, 100.0, 100.0, "cube", 2000.0, 0.0, 101, 301, 201)
C2 = Workload("C2", 1000, 4, 80.0, 120.0, "cube", 0.0, 0.2, 102, 302, 202)
C3 = Workload("C3", 10_000, 3, 100.0, 100.0, "slab", 20_000.0, 0.3, 103, 303, 203)
C4 = Workload("C4", 100_000, 3, 100.0, 100.0, "slab", 60_000.0, 0.3, 104, 304, 204)
C5 = Workload("C5", 10_000, 4, 90.0, 110.0, "slab", 20_000.0, 0.3, 105, 305, 205)
CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5)}


def scaled(w: Workload, N: int, name: str | None = None) -> Workload:
    """Same recipe with fewer spheres; a slab keeps its filling fraction and aspect by shrinking laterally
    (lateral ~ sqrt(N)) so that its thickness stays that of the full-size config."""
    lateral = w.lateral_nm
    if w.shape == "slab":
        lateral = w.lateral_nm * np.sqrt(N / w.N)
    return Workload(name or f"{w.name}_N{N}", N, w.lmax, w.radius_lo, w.radius_hi, w.shape, lateral, w.filling,
                    w.seed_pos, w.seed_rad, w.seed_b)


def radii(w: Workload) -> np.ndarray:
    if w.radius_lo == w.radius_hi:
        return np.full(w.N, w.radius_lo, dtype=np.float64)
    return np.random.default_rng(w.seed_rad).uniform(w.radius_lo, w.radius_hi, w.N)


def box(w: Workload, rad: np.ndarray) -> np.ndarray:
    """Edge lengths of the box that contains the sphere CENTRES."""
    vol = float(np.sum(4.0 / 3.0 * np.pi * rad**3))
    if w.shape == "cube":
        edge = w.lateral_nm if w.filling == 0.0 else (vol / w.filling) ** (1.0 / 3.0)
        return np.array([edge, edge, edge])
    thickness = vol / (w.filling * w.lateral_nm**2)
    return np.array([w.lateral_nm, w.lateral_nm, thickness])


def rsa_positions(rad: np.ndarray, edges: np.ndarray, seed: int, gap: float = GAP_NM,
                  max_trials: int = 50_000_000) -> np.ndarray:
    """Random sequential addition: sphere i is offered uniformly random centres in the box until one keeps
    |r_i - r_j| >= R_i + R_j + gap for every sphere j placed before; spheres are placed in index order.
    A uniform grid with at most one centre per cell makes each trial O(1).  Candidates are drawn in batches
    from one default_rng(seed) stream; a batch is pre-filtered against the spheres placed before it
    (vectorised) and the survivors are then offered one by one, which gives exactly the sequential result."""
    rng = np.random.default_rng(seed)
    N = rad.shape[0]
    pos = np.zeros((N, 3), dtype=np.float64)
    dmin = 2.0 * float(rad.min()) + gap
    cell = dmin / np.sqrt(3.0) * 0.999                      # cell diagonal < dmin: one centre per cell
    ncell = np.maximum(1, np.ceil(edges / cell).astype(np.int64))
    reach = int(np.ceil((2.0 * float(rad.max()) + gap) / cell))
    pad = reach
    grid = np.full(tuple(ncell + 2 * pad), -1, dtype=np.int64)
    offs = np.stack(np.meshgrid(*([np.arange(-reach, reach + 1)] * 3), indexing="ij"), axis=-1).reshape(-1, 3)
    placed, trials = 0, 0
    while placed < N:
        if trials > max_trials:
            raise RuntimeError(f"RSA jammed: {placed} of {N} placed after {trials} trials")
        B = int(min(max(256, (N - placed)), 65536))
        cand = rng.random((B, 3)) * edges
        trials += B
        cidx = np.minimum((cand / cell).astype(np.int64), ncell - 1) + pad
        # vectorised pre-filter against everything placed before this batch, for the radius of the
        # sphere that would be placed NEXT is not known per candidate -> use the smallest admissible
        # distance (conservative: only rejects what any sphere would reject), exact test below.
        nb = grid[cidx[:, None, 0] + offs[None, :, 0], cidx[:, None, 1] + offs[None, :, 1],
                  cidx[:, None, 2] + offs[None, :, 2]]                     # [B, n_off]
        has = nb >= 0
        nbc = np.where(has, nb, 0)
        dist2 = np.sum((cand[:, None, :] - pos[nbc]) ** 2, axis=-1)
        lim = (float(rad.min()) + rad[nbc] + gap) ** 2
        ok = ~np.any(has & (dist2 < lim), axis=1)
        for c in np.nonzero(ok)[0]:
            if placed >= N:
                break
            ci = cidx[c]
            sl = grid[ci[0] - reach:ci[0] + reach + 1, ci[1] - reach:ci[1] + reach + 1,
                      ci[2] - reach:ci[2] + reach + 1]
            j = sl[sl >= 0]
            if j.size:
                d2 = np.sum((pos[j] - cand[c]) ** 2, axis=1)
                if np.any(d2 < (rad[placed] + rad[j] + gap) ** 2):
                    continue
            pos[placed] = cand[c]
            grid[ci[0], ci[1], ci[2]] = placed
            placed += 1
    return pos


def positions(w: Workload) -> tuple[np.ndarray, np.ndarray]:
    """(pos [N,3] nm, radii [N] nm) of a workload; centres are shifted so the box is centred on the origin
    in x and y and starts at z = 0."""
    rad = radii(w)
    edges = box(w, rad)
    pos = rsa_positions(rad, edges, w.seed_pos)
    pos[:, 0] -= edges[0] / 2
    pos[:, 1] -= edges[1] / 2
    return pos, rad


def gaussian_coefficients(N: int, nmax: int, seed: int) -> np.ndarray:
    """b ~ CN(0,1): Re, Im i.i.d. N(0, 1/2) in FP64, rounded ONCE to complex64 (reading R18); both the CUDA
    path and the oracle (promoting to FP64) read these rounded values."""
    rng = np.random.default_rng(seed)
    z = rng.normal(0.0, np.sqrt(0.5), (N, nmax)) + 1j * rng.normal(0.0, np.sqrt(0.5), (N, nmax))
    return z.astype(np.complex64)


def sample_receivers(N: int, count: int, seed: int) -> np.ndarray:
    """`count` distinct receiver indices chosen by default_rng(seed), sorted."""
    return np.sort(np.random.default_rng(seed).choice(N, size=min(count, N), replace=False)).astype(np.int64)


def min_gap(pos: np.ndarray, rad: np.ndarray) -> float:
    """Smallest surface-to-surface distance (O(N^2) memory-light loop; for tests on small N)."""
    best = np.inf
    for i in range(pos.shape[0] - 1):
        d = np.sqrt(np.sum((pos[i + 1:] - pos[i]) ** 2, axis=1)) - rad[i + 1:] - rad[i]
        best = min(best, float(d.min()))
    return best
