"""celes_far_field_noalloc (include/celes.h): the far field for callers that must not allocate -- its tables live in one
static device array of the library instead of cudaMalloc'ed scratch.  Checked against the existing celes_far_field on
calls in a row that share (and overwrite) that array.  Named so that pytest collects it LAST; passes alone in a fresh
process and after the other tests."""
import dataclasses

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import paper_1706_02145_b200 as celes
from paper_1706_02145_b200 import fields, workloads
from oracle import celes_oracle as orc

pytestmark = pytest.mark.gpu

FIELD_TOL = 1e-4        # the far-field tests' bound: worst component within 1e-4 of the largest one


def directions(n, seed):
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.uniform(0, 2 * np.pi, n)), np.ascontiguousarray(np.arccos(rng.uniform(-1, 1, n)))


def close(g, ref):
    g, ref = g.cpu().numpy(), ref.cpu().numpy() if hasattr(ref, "cpu") else np.asarray(ref)
    return float(np.abs(g - ref).max() / np.abs(ref).max())


@pytest.mark.parametrize("lmax", [3, 4])
def test_far_field_noalloc_matches_the_existing_path_on_calls_in_a_row(lmax):
    w = dataclasses.replace(workloads.scaled(workloads.C3, 2000), lmax=lmax)
    pos, rad = workloads.positions(w)
    ctx = celes.celes_setup(pos, rad, fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE), w.k, w.lmax)
    b_host = workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)
    b = torch.from_numpy(b_host).cuda()
    sets = [directions(1500, 1), directions(37, 2)]                   # ragged counts, very different sizes
    out = [torch.full((a.size, 2), 7.0 + 7.0j, dtype=torch.complex64, device="cuda") for a, _ in sets]
    # the no-allocation entry point FIRST: this context's own (lazily allocated) scratch does not exist yet
    for (al, be), g in zip(sets, out):
        celes.celes_far_field_noalloc(ctx, b, al, be, g)
    torch.cuda.synchronize()
    ref = [celes.celes_far_field(ctx, b, al, be).clone() for al, be in sets]      # the existing path
    for g, r in zip(out, ref):
        assert close(g, r) <= FIELD_TOL
    # and against the oracle for the small set (independent of both GPU paths)
    al, be = sets[1]
    assert close(out[1], orc.far_field_amplitude(pos, w.k, w.lmax, b_host, al, be)) <= FIELD_TOL
    # again in the other order, on the array the calls above left full: 37 directions over 1500 directions' leftovers,
    # then 1500 again, each into a cleared output
    for k in (1, 0, 1):
        out[k].zero_()
        celes.celes_far_field_noalloc(ctx, b, sets[k][0], sets[k][1], out[k])
        assert close(out[k], ref[k]) <= FIELD_TOL
    # a second context (other coefficients) shares the same array: interleaved calls on one stream stay correct
    b2 = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, 99)).cuda()
    g2 = torch.empty(37, 2, dtype=torch.complex64, device="cuda")
    celes.celes_far_field_noalloc(ctx, b2, al, be, g2)
    celes.celes_far_field_noalloc(ctx, b, al, be, out[1])
    assert close(g2, celes.celes_far_field(ctx, b2, al, be)) <= FIELD_TOL and close(out[1], ref[1]) <= FIELD_TOL


def test_far_field_noalloc_limit_and_no_device_allocation():
    w = workloads.scaled(workloads.C3, 600)
    pos, rad = workloads.positions(w)
    ctx = celes.celes_setup(pos, rad, fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE), w.k, w.lmax)
    b = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)).cuda()
    nmax_dir = celes.CELES_FAR_FIELD_NOALLOC_MAX_DIR
    # beyond the stated maximum: a clear error of its own, nothing launched, the output untouched
    al, be = directions(nmax_dir + 1, 3)
    g = torch.full((nmax_dir + 1, 2), 5.0 - 3.0j, dtype=torch.complex64, device="cuda")
    with pytest.raises(celes.CelesError) as e:
        celes.celes_far_field_noalloc(ctx, b, al, be, g)
    assert e.value.code == celes.CELES_ELIMIT and "capacity" in str(e.value)
    torch.cuda.synchronize()
    assert bool((g == (5.0 - 3.0j)).all())
    # exactly the maximum works, twice in a row, and the calls take no device memory: free memory does not go down
    # (the existing path would have to grow its scratch for this many directions)
    al, be = directions(nmax_dir, 4)
    g = torch.empty(nmax_dir, 2, dtype=torch.complex64, device="cuda")
    first = torch.empty_like(g)                                       # every tensor exists before the measurement
    celes.celes_far_field_noalloc(ctx, b, al, be, g)                  # first use of these kernels (module load)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    celes.celes_far_field_noalloc(ctx, b, al, be, g)
    first.copy_(g)
    celes.celes_far_field_noalloc(ctx, b, al, be, g)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    assert torch.equal(torch.view_as_real(g), torch.view_as_real(first))          # same inputs, same array: same bits
    assert close(g, celes.celes_far_field(ctx, b, al, be)) <= FIELD_TOL
