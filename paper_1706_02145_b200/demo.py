"""End-to-end example of the C ABI through the Python binding (needs a B200; there is no CPU fallback):

    python -m paper_1706_02145_b200.demo [--n 2000] [--lmax 3] [--out gpurun_out/demo]

A slab of N spheres (recipe of BASELINE.json config 3, scaled) is illuminated by a plane wave travelling along +z,
polarised along x; eq. (8) is solved with GMRES(30); the total field |E_in + E_scat| is mapped on the
plane y = 0 outside the spheres (eq. 3, the picture of Figs. 2 and 6; pixels inside a
sphere are set to 0: the internal field is not part of this library), and the far-field intensity sum_j |g_j|^2 of
(D.3) on a (beta, alpha) grid.  Both arrays are written as .npy and as 8-bit .pgm images (no graphics stack needed).
"""
from __future__ import annotations

import argparse
import os

import numpy as np


def write_pgm(path: str, a: np.ndarray) -> None:
    a = np.asarray(a, dtype=np.float64)
    hi = float(a.max()) or 1.0
    img = np.clip(255.0 * a / hi, 0, 255).astype(np.uint8)
    with open(path, "wb") as f:
        f.write(b"P5\n%d %d\n255\n" % (img.shape[1], img.shape[0]))
        f.write(img.tobytes())


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=2000)
    ap.add_argument("--lmax", type=int, default=3)
    ap.add_argument("--pixels", type=int, default=384)
    ap.add_argument("--out", default=os.path.join("gpurun_out", "demo"))
    args = ap.parse_args()

    import dataclasses
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, workloads

    w = dataclasses.replace(workloads.scaled(workloads.C3, args.n), lmax=args.lmax)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax)
    a_in = celes.celes_plane_wave(ctx, 0.0, 0.0, 2)                 # +z, x-polarised (A.13)
    b = torch.zeros(w.N, w.nmax, dtype=torch.complex64, device="cuda")
    info = celes.celes_solve(ctx, a_in, b, restart=30, rtol=1e-4, max_iters=2000)
    print(f"solve: {info['iterations']} iterations, {info['matvecs']} matvecs, residual {info['rel_residual']:.2e}, "
          f"{info['seconds']:.3f} s")

    # near field on the plane y = 0
    n = args.pixels
    half = 0.5 * (pos[:, 0].max() - pos[:, 0].min())
    xs = np.linspace(-half, half, n)
    zs = np.linspace(pos[:, 2].min() - 1500.0, pos[:, 2].max() + 2500.0, n)
    Z, X = np.meshgrid(zs, xs, indexing="ij")
    pts = np.stack([X.ravel(), np.zeros(n * n), Z.ravel()], axis=1)
    inside = np.zeros(n * n, dtype=bool)
    near = np.abs(pos[:, 1]) < rad                                # spheres cut by the plane
    for c, r in zip(pos[near], rad[near]):
        inside |= np.sum((pts - c) ** 2, axis=1) < r * r
    E = celes.celes_scattered_field(ctx, b, pts).cpu().numpy().astype(np.complex128)
    E[:, 0] += np.exp(1j * w.k * pts[:, 2])                       # incident plane wave, x-polarised
    mag = np.sqrt(np.sum(np.abs(E) ** 2, axis=1))
    mag[inside] = 0.0
    mag = mag.reshape(n, n)

    # far-field intensity
    nb = 180
    beta = (np.arange(nb) + 0.5) * np.pi / nb
    alpha = np.arange(2 * nb) * np.pi / nb
    B, A = np.meshgrid(beta, alpha, indexing="ij")
    g = celes.celes_far_field(ctx, b, A.ravel(), B.ravel()).cpu().numpy()
    inten = np.sum(np.abs(g) ** 2, axis=1).reshape(nb, 2 * nb)

    os.makedirs(args.out, exist_ok=True)
    np.save(os.path.join(args.out, "near_field_abs_E.npy"), mag)
    np.save(os.path.join(args.out, "far_field_intensity.npy"), inten)
    write_pgm(os.path.join(args.out, "near_field_abs_E.pgm"), mag)
    write_pgm(os.path.join(args.out, "far_field_intensity.pgm"), np.log10(1.0 + inten / inten.max() * 1e4))
    print(f"|E| on y = 0: min {mag[~inside.reshape(n, n)].min():.3f}, max {mag.max():.3f}; far-field peak at beta = "
          f"{np.degrees(beta[np.unravel_index(inten.argmax(), inten.shape)[0]]):.1f} deg; written to {args.out}/")


if __name__ == "__main__":
    main()
