"""Receiver-sharded coupling product across ranks (last clause): rank r owns the receiver rows
[row_begin, row_end) of y = W b and the matching rows of b; one all-gather of b per product gives every rank the full
emitter vector, then celes_coupling_matvec_rows (include/celes.h) computes the rank's rows.  No other collective: the
rows of y stay where they are needed next (the Krylov vectors of a sharded solve are row-sharded too).

north_star fixes ONE GPU, so this is an optional deployment mode (bench.py --shard receivers), not the default; the
paper itself is single-GPU.  The arithmetic is the library's: this module only cuts index ranges and
calls torch.distributed.
"""
from __future__ import annotations

import numpy as np


def row_slices(N: int, world: int, align: int = 1) -> list[tuple[int, int]]:
    """world contiguous row ranges covering [0, N), sizes within one `align` unit of each other, boundaries on multiples
    of `align` (the receiver-block size keeps every receiver block on one rank; any boundary is valid for the library)."""
    if N < 1 or world < 1 or align < 1:
        raise ValueError("row_slices: N, world, align >= 1")
    units = (N + align - 1) // align
    cuts = [min(N, ((units * r) // world) * align) for r in range(world)] + [N]
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def all_gather_rows(b_rows, slices, rank: int, group=None):
    """Full [N, nmax] tensor from every rank's rows (ranks may own different numbers of rows, empty ones included).
    One collective: all_gather on equal-sized padded pieces."""
    import torch
    import torch.distributed as dist
    world = len(slices)
    nmax = b_rows.shape[1]
    r0, r1 = slices[rank]
    if b_rows.shape[0] != r1 - r0:
        raise ValueError("all_gather_rows: b_rows must hold this rank's rows")
    longest = max(e - s for s, e in slices)
    piece = torch.zeros(longest, nmax, dtype=b_rows.dtype, device=b_rows.device)
    piece[: r1 - r0] = b_rows
    out = torch.empty(world * longest, nmax, dtype=b_rows.dtype, device=b_rows.device)
    if world == 1:
        out.copy_(piece)
    else:
        # complex dtypes travel as their real view (same bytes)
        dist.all_gather_into_tensor(torch.view_as_real(out) if out.is_complex() else out,
                                    torch.view_as_real(piece) if piece.is_complex() else piece, group=group)
    if all(e - s == longest for s, e in slices):
        return out
    return torch.cat([out[r * longest: r * longest + (e - s)] for r, (s, e) in enumerate(slices)], dim=0)


def sharded_coupling_matvec(ctx, b_rows, slices, rank: int, y_rows=None, group=None, system: bool = False):
    """Rows [slices[rank]) of W b (system: of b - T W b) from this rank's rows of b."""
    from . import binding
    b_full = all_gather_rows(b_rows, slices, rank, group)
    r0, r1 = slices[rank]
    fn = binding.celes_system_matvec_rows if system else binding.celes_coupling_matvec_rows
    return fn(ctx, r0, r1, b_full, y_rows)
