#!/usr/bin/env python3
"""bench.py -- coupling-matvec throughput of the CELES hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4|C3] [--impl ours|reference]

A step is one pass of the whole hot path y = W b (pack -> coupling kernel -> finalize) over the synthetic
ensemble of BASELINE.json config 4 (N = 1e5 spheres, lmax = 3).  `value` is sphere-pair
translations per second, N (N-1) / time, inputs resident in HBM; `e2e` is the same metric through
celes_coupling_matvec_host with pinned HOST buffers (H2D + D2H inside the timed region).

The path does not shard (north_star: one GPU, no collectives): --gpus N runs N independent replicas
("replicas only"), value = pairs of all replicas / max-over-ranks time.  --shard receivers is the
optional receiver-sharded mode of SURVEY.md 8(e) (one all-gather of b per product, strong scaling).

--impl reference times the FP64 CPU oracle (oracle/), as it stands, on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sphere_pair_translations_per_s"
UNIT = "pairs/s"
# FP32 flops and FMA-pipe lane operations per ordered pair are COUNTED in the SASS of the built library's coupling
# kernel (paper_1706_02145_b200/sass_count.py: opcode histogram of the per-pair loop body; flops = 4 FFMA2 + 2 (FMUL2 +
# FADD2) + 2 FFMA + FMUL + FADD, lane ops = 2 per packed instruction + 1 per scalar one).  The FMA
# pipe retires 128 lane operations per SM per clock whatever their kind, so lane_ops x pairs / (128 x SMs x clock x
# time) is the pipe utilisation, while the flop fraction also charges every multiply / add as half an FMA.
FP32_LANES_PER_SM = 128
PRECOND_EDGE_NM = 600.0     # lateral cuboid edge of the preconditioned config-5 solve in the default line
# dram__bytes_read.sum + dram__bytes_write.sum of one coupling-kernel launch, from the ncu --set full capture
# summarised in the named file under profiles/ (a capture, not a live measurement: ncu cannot run inside the timed run)
NCU_DRAM_BYTES_PER_LAUNCH = {("C4", "rotated"): (87.3e6, "profiles/r02i_kernel_c4.md")}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--translation", default="rotated", choices=["rotated", "direct"])
    ap.add_argument("--solve", action="store_true",
                    help="time celes_solve (plane wave, GMRES(30), rtol 1e-4) on the workload instead (config 5: --workload C5)")
    ap.add_argument("--precond-edge", type=float, default=0.0,
                    help="with --solve: lateral edge (nm) of the cuboids of the block-diagonal preconditioner (0 = none)")
    ap.add_argument("--far-field", type=int, default=0, metavar="NB",
                    help="time celes_far_field on NB x 2NB directions (Gauss-Legendre x uniform azimuth) instead")
    ap.add_argument("--near-field", type=int, default=0, metavar="NP",
                    help="time celes_scattered_field on an NP x NP grid of points in the plane 300 nm above the slab instead")
    ap.add_argument("--gaussian-beam", action="store_true",
                    help="time celes_gaussian_beam (waist 4 um, PAPER.md:140, centred on the slab, normal incidence) instead")
    ap.add_argument("--levels", type=int, default=0,
                    help="levels of the guided work partition (celes_options.levels; 0 = library default)")
    ap.add_argument("--lmax", type=int, default=0, help="override the workload's truncation order (1..5)")
    ap.add_argument("--hankel", default="registers", choices=["registers", "table"],
                    help="h_p(kd) in registers (default) or from the paper's lookup table (PAPER.md:130)")
    ap.add_argument("--method", default="gmres", choices=["gmres", "bicgstab"], help="with --solve")
    ap.add_argument("--restart", type=int, default=30, help="with --solve: GMRES restart length (BASELINE config 5: 30)")
    ap.add_argument("--cta-trace", action="store_true",
                    help="per-CTA start / end times and SM of the coupling kernel for --levels 1 and the default partition "
                         "(needs a library built with CELES_NVCC_EXTRA=-DCELES_TRACE python -m paper_1706_02145_b200.build --force)")
    ap.add_argument("--shard", default="none", choices=["none", "receivers"],
                    help="with --gpus N > 1: 'receivers' shards the receiver rows over the ranks (one all-gather of b per "
                         "product, strong scaling; SURVEY.md 8(e)) instead of running N replicas (the default, north_star)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="CPU work of the cpu_baseline sample")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (the profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=f, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                p = [x.strip() for x in line.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1])); mx.append(float(p[2])); pw.append(float(p[3]))
                except ValueError:
                    continue
                for nm, v in zip(names, p[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(pw)))
        return out


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        return {}


def device_sm_clock_hz(index: int = 0) -> float:
    """Maximum SM clock of the device (nvidia-smi clocks.max.sm; MEASURED_PEAKS.json if the query fails)."""
    try:
        out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", str(index)],
                             capture_output=True, text=True, timeout=20).stdout
        return float(out.strip().splitlines()[0]) * 1e6
    except (OSError, ValueError, IndexError, subprocess.TimeoutExpired):
        return float(measured_peaks().get("sm_max_mhz", 1965.0)) * 1e6


def max_over_ranks(value: float, world: int, device) -> float:
    """Slowest rank's value (replicas only: no data-path collective; this all-reduce of one
    scalar is the measurement, not the method).  Works with nccl (CUDA tensor) and gloo (CPU tensor)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(pairs_per_replica: int, steps: int, world: int, slowest_total_ms: float) -> float:
    """Whole-job pair translations per second of `world` independent replicas timed by the slowest one."""
    return world * pairs_per_replica * steps / (slowest_total_ms * 1e-3)


def oracle_sample_rate(w, pos, b, seconds: float):
    """Times the oracle (as it stands) on whole receivers of workload w until about `seconds` of CPU work."""
    from oracle import celes_oracle as orc
    from paper_1706_02145_b200 import workloads
    t0 = time.perf_counter()
    orc.coupling_matvec(pos, w.k, w.lmax, b, receivers=np.array([0]))          # calibration: one receiver
    t1 = time.perf_counter() - t0
    cores = max(1, orc.LAST_THREADS)
    per_recv = t1                                                             # one receiver is one thread's work
    n_recv = int(max(cores, min(w.N, seconds / max(per_recv, 1e-9) * cores)))
    n_recv = (n_recv // cores) * cores
    recv = workloads.sample_receivers(w.N, n_recv, 404)
    t0 = time.perf_counter()
    orc.coupling_matvec(pos, w.k, w.lmax, b, receivers=recv)
    dt = time.perf_counter() - t0
    pairs = len(recv) * (w.N - 1)
    return pairs / dt, cores, len(recv), dt


def run_reference(args, w):
    """--impl reference: the oracle on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import celes_oracle as orc
    from paper_1706_02145_b200 import workloads
    pos, rad = workloads.positions(w)
    b = workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)
    t0 = time.perf_counter()
    orc.coupling_matvec(pos, w.k, w.lmax, b, receivers=np.array([0]))
    per_recv = time.perf_counter() - t0
    cores = max(1, orc.LAST_THREADS)
    budget = 150.0 / max(1, args.steps + args.warmup)                         # seconds per step
    n_recv = int(max(cores, min(w.N, budget / max(per_recv, 1e-9) * cores)))
    n_recv = max(cores, (n_recv // cores) * cores)
    recv = workloads.sample_receivers(w.N, n_recv, 404)
    for _ in range(args.warmup):
        orc.coupling_matvec(pos, w.k, w.lmax, b, receivers=recv)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.coupling_matvec(pos, w.k, w.lmax, b, receivers=recv)
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    value = len(recv) * (w.N - 1) / dt
    sample = f"{len(recv)} seeded receivers x {w.N - 1} emitters per step (full emitter sum each)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax} slab RSA ff=0.3 (sampled receivers)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def precond_apply_roofline(celes, ctx, v, pc, reps: int = 20):
    """The HBM-bound kernel of the preconditioner, z = blockdiag(M_j^{-1}) v: CUDA-event time per application and the
    achieved bandwidth (stored blocks + the two vectors) against the measured copy bandwidth of MEASURED_PEAKS.json."""
    import torch
    z = torch.empty_like(v)
    for _ in range(3):
        celes.celes_precond_apply(ctx, v, z)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        celes.celes_precond_apply(ctx, v, z)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    nbytes = pc["block_bytes"] + 2 * v.numel() * 8
    peaks = measured_peaks()
    peak = peaks.get("hbm_gbs", 6650.0)
    return {"bound": "hbm", "ms": ms, "bytes": nbytes, "achieved": nbytes / ms / 1e6, "peak": peak, "unit": "GB/s",
            "frac": nbytes / ms / 1e6 / peak, "peak_kind": "measured (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback",
            "note": "blocks larger than L2 are re-read from HBM every application"}


def run_solve(args, w):
    """BASELINE.json config 5: time to solution and iteration count of celes_solve; one JSON line."""
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, workloads
    torch.cuda.set_device(0)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax, translation=args.translation)
    a_in = torch.from_numpy(fields.plane_wave_coefficients(pos, w.k, w.lmax).astype(np.complex64)).cuda()
    x = torch.zeros(w.N, w.nmax, dtype=torch.complex64, device="cuda")
    celes.celes_solve(ctx, a_in, x, restart=args.restart, rtol=1e-4, max_iters=3)          # warm-up (allocations, caches)
    pc = None
    if args.precond_edge > 0:
        celes.celes_precond_setup(ctx, [args.precond_edge, args.precond_edge, 0.0])   # warm-up (kernel load)
    runs = []
    for _ in range(max(1, args.steps)):
        x.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if args.precond_edge > 0:                                                # set-up is part of the time to solution
            pc = celes.celes_precond_setup(ctx, [args.precond_edge, args.precond_edge, 0.0])
        info = celes.celes_solve(ctx, a_in, x, restart=args.restart, rtol=1e-4, max_iters=2000, precond=pc is not None,
                                 method=args.method)
        torch.cuda.synchronize()
        runs.append((time.perf_counter() - t0, info))
    secs = [r[0] for r in runs]
    info = runs[-1][1]
    pc_line = None if pc is None else precond_apply_roofline(celes, ctx, a_in, pc)
    print(json.dumps({
        "metric": "time_to_solution_s", "value": float(np.median(secs)), "unit": "s", "n_gpus": 1, "steps": len(runs),
        "warmup": 1, "higher_is_better": False, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax} plane wave +z x-pol, GMRES({args.restart}) rtol 1e-4",
                   "translation": args.translation, "method": args.method,
                   "preconditioner": None if pc is None else dict(pc, edge_nm=args.precond_edge)},
        "precond_apply_roofline": pc_line,
        "iterations": info["iterations"], "matvecs": info["matvecs"], "converged": info["converged"],
        "rel_residual": info["rel_residual"], "seconds_all": secs,
        "ms_per_matvec_incl_krylov": 1e3 * float(np.median(secs)) / max(1, info["matvecs"])}))


def run_far_field(args, w):
    """celes_far_field on the workload: time per call, (direction, polarisation, sphere) terms per second."""
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, workloads
    torch.cuda.set_device(0)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax)
    b = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)).cuda()
    nb = args.far_field
    xb, _ = np.polynomial.legendre.leggauss(nb)
    A, B = np.meshgrid(2 * np.pi * np.arange(2 * nb) / (2 * nb), np.arccos(xb), indexing="ij")
    al, be = A.ravel(), B.ravel()
    g = torch.empty(al.size, 2, dtype=torch.complex64, device="cuda")
    for _ in range(max(3, args.warmup)):
        celes.celes_far_field(ctx, b, al, be, g)
    times = []
    for _ in range(max(1, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        celes.celes_far_field(ctx, b, al, be, g)          # asynchronous: direction upload + coefficient, sum and reduce kernels
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e-3)
    sec = float(np.median(times))
    terms = 2.0 * al.size * w.N
    # FMA-pipe lane operations that every (direction, polarisation, sphere) term certainly executes: 2 nmax FFMA2 of the
    # packed sums + 3 FADD2 + 2 FFMA2 of the combine / accumulate.  The phase (FP64), its reduction and the sine / cosine
    # are shared by the two polarisations of a direction at lmax <= 3 and are NOT counted: a lower bound on the busy pipe.
    lane = 4.0 * w.nmax + 10.0
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    print(json.dumps({
        "metric": "far_field_terms_per_s", "value": terms / sec, "unit": "(direction,polarisation,sphere)/s", "n_gpus": 1,
        "steps": len(times), "ms_per_call": sec * 1e3, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax}", "directions": int(al.size)},
        "roofline": {"bound": "alu", "lane_ops_per_term": lane, "counted": "packed sums + accumulate only (lower bound)",
                     "fma_pipe_utilisation_whole_call": lane * terms / sec / (FP32_LANES_PER_SM * sm * device_sm_clock_hz())}}))


def run_gaussian_beam(args, w):
    """celes_gaussian_beam (Appendix C, (C.7)-(C.8)): initial-field coefficients of the paper's beam (waist 4 um,
    PAPER.md:140) for every sphere of the workload; FP64 input preparation, once per simulation."""
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, workloads
    torch.cuda.set_device(0)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax)
    centre = [0.0, 0.0, float(pos[:, 2].min()) - 200.0]
    a_in = torch.empty(w.N, w.nmax, dtype=torch.complex64, device="cuda")
    for _ in range(max(2, args.warmup)):
        celes.celes_gaussian_beam(ctx, 4000.0, centre, a_in=a_in)
    times = []
    for _ in range(max(1, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        celes.celes_gaussian_beam(ctx, 4000.0, centre, a_in=a_in)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e-3)
    sec = float(np.median(times))
    print(json.dumps({
        "metric": "beam_coefficients_per_s", "value": w.N * w.nmax / sec, "unit": "coefficients/s", "n_gpus": 1,
        "steps": len(times), "ms_per_call": sec * 1e3, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax}", "waist_nm": 4000.0,
                   "norm_a_in": float(torch.linalg.vector_norm(a_in))}}))


def run_sharded(args, w):
    """--gpus N --shard receivers under torchrun: every rank owns a slice of the receiver rows (and of b); a step is one
    all-gather of b (NCCL) + celes_coupling_matvec_rows on the rank's rows.  value = N (N - 1) / slowest rank's time:
    total work is fixed, scaling = strong.  Not the default: north_star is one GPU."""
    import torch
    import torch.distributed as dist
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, sharding, workloads
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax, translation=args.translation)
    slices = sharding.row_slices(w.N, world, celes.celes_work_partition(ctx)["receivers_per_block"])
    r0, r1 = slices[rank]
    b_rows = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)[r0:r1]).cuda()
    y_rows = torch.empty_like(b_rows)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        sharding.sharded_coupling_matvec(ctx, b_rows, slices, rank, y_rows)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev = []
    for _ in range(args.steps):
        flush.zero_()
        a, c = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        sharding.sharded_coupling_matvec(ctx, b_rows, slices, rank, y_rows)
        c.record()
        ev.append((a, c))
    barrier()
    clocks = sampler.stop()
    total_ms = max_over_ranks(float(sum(a.elapsed_time(c) for a, c in ev)), world, "cuda")
    pairs = w.N * (w.N - 1)
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": pairs * args.steps / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax}", "pairs_per_step": pairs,
                       "parallelism": f"receiver rows sharded over {world} ranks, all-gather of b per product",
                       "rows_per_rank": [e - s for s, e in slices],
                       "l2": "flushed between timed iterations (256 MiB write)"},
            "clocks": clocks, "gpu_launches": 3 * args.steps}))
    if world > 1:
        dist.destroy_process_group()


def run_near_field(args, w):
    """celes_scattered_field (eq. 3) on NP x NP points of a plane above the slab: time per call and
    (point, sphere) terms per second."""
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, workloads
    torch.cuda.set_device(0)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax)
    b = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)).cuda()
    npts = args.near_field
    lo, hi = pos.min(axis=0), pos.max(axis=0)
    X, Y = np.meshgrid(np.linspace(lo[0], hi[0], npts), np.linspace(lo[1], hi[1], npts), indexing="ij")
    pts = np.stack([X.ravel(), Y.ravel(), np.full(X.size, hi[2] + rad.max() + 300.0)], axis=1)
    for _ in range(max(2, args.warmup)):
        celes.celes_scattered_field(ctx, b, pts)
    times = []
    for _ in range(max(1, args.steps)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        celes.celes_scattered_field(ctx, b, pts)
        e1.record()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1) * 1e-3)
    sec = float(np.median(times))
    terms = float(pts.shape[0]) * w.N
    print(json.dumps({
        "metric": "near_field_terms_per_s", "value": terms / sec, "unit": "(point,sphere)/s", "n_gpus": 1,
        "steps": len(times), "ms_per_call": sec * 1e3, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax}", "points": int(pts.shape[0])}}))


def run_cta_trace(args, w):
    """Diagnostic build only: how long every CTA of the coupling kernel ran and on which SM (globaltimer, %smid), for
    one wave of equal runs (levels = 1) and for the default guided partition.  One JSON line per partition."""
    import ctypes
    import torch
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import binding, fields, workloads
    L = binding.lib()
    if not hasattr(L, "celes_debug_trace"):
        raise SystemExit("--cta-trace: rebuild with CELES_NVCC_EXTRA=-DCELES_TRACE python -m paper_1706_02145_b200.build --force")
    L.celes_debug_trace.argtypes = [ctypes.c_void_p]
    torch.cuda.set_device(0)
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    b = torch.from_numpy(workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b)).cuda()
    y = torch.empty_like(b)
    for levels in (1, 0):
        ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax, levels=levels)
        for _ in range(3):
            celes.celes_coupling_matvec(ctx, b, y)
        torch.cuda.synchronize()
        raw = np.zeros(3 * 8192, dtype=np.uint64)
        assert L.celes_debug_trace(raw.ctypes.data) == 0
        n = min(8192, celes.celes_work_partition(ctx)["ctas"])
        t = raw.reshape(-1, 3)[:n].astype(np.int64)
        start, end = (t[:, 1] - t[:, 1].min()) / 1e3, (t[:, 2] - t[:, 1].min()) / 1e3
        dur = end - start
        per_sm = {}
        for s, d in zip(t[:, 0], dur):
            per_sm.setdefault(int(s), []).append(float(d))
        busy = np.array([sum(v) for v in per_sm.values()])
        first = dur[:len(per_sm) * 2] if levels == 1 else dur
        print(json.dumps({
            "workload": w.name, "levels": levels or "default", "ctas": int(n), "sms": len(per_sm), "kernel_us": float(end.max()),
            "cta_us": {"min": float(dur.min()), "median": float(np.median(dur)), "max": float(dur.max())},
            "per_sm_busy_us": {"min": float(busy.min()), "max": float(busy.max())},
            "ctas_per_sm": {"min": min(len(v) for v in per_sm.values()), "max": max(len(v) for v in per_sm.values())},
            "last_start_us": float(start.max()),
            "faster_of_two_resident_ctas_finishes_at": float(np.median([min(v) / max(v) for v in per_sm.values() if len(v) == 2]))
            if levels == 1 and len(first) else None}))
        del ctx


def time_coupling(celes, ctx, b, y, steps, flush, stream):
    """CUDA-event times (ms) of `steps` coupling matvecs on `stream`, L2 flushed before each (outside the events)."""
    import torch
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, c in ev:
        flush.zero_()
        a.record(stream)
        celes.celes_coupling_matvec(ctx, b, y)
        c.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(c) for a, c in ev]


def alu_roofline(counts, pairs, ms, sm_count, sm_max_mhz, sm_mhz):
    """Roofline numbers of one coupling launch from the SASS-counted work per pair (sass_count.py)."""
    achieved = counts["flops_per_pair"] * pairs / (ms * 1e-3)
    lane_rate = counts["lane_ops_per_pair"] * pairs / (ms * 1e-3)
    nominal = 2.0 * FP32_LANES_PER_SM * sm_count * sm_max_mhz * 1e6
    return {"bound": "alu", "achieved": achieved / 1e12, "peak": nominal / 1e12, "unit": "TFLOP/s",
            "frac": achieved / nominal,
            "peak_kind": "derived: 2 x 128 FP32 lanes x SMs x clocks.max.sm (DESIGN.md section 6)",
            "frac_of_peak_at_observed_clock": achieved / (2.0 * FP32_LANES_PER_SM * sm_count * sm_mhz * 1e6),
            "flops_per_pair": counts["flops_per_pair"], "lane_ops_per_pair": counts["lane_ops_per_pair"],
            "fp32_opcodes_per_pair": counts["fp32"], "packed_non_fma_per_pair": counts["packed_non_fma"],
            "counts_source": counts["source"],
            "fma_pipe_utilisation": lane_rate / (FP32_LANES_PER_SM * sm_count * sm_mhz * 1e6)}


def solve_c5(celes, fields, workloads, translation, precond_edge=0.0):
    """BASELINE.json config 5 (N = 1e4, lmax = 4, plane wave +z x-pol, GMRES(30), rtol 1e-4): wall-clock time to
    solution (preconditioner set-up included when one is used), iterations, matvecs, true relative residual."""
    import torch
    w = workloads.CONFIGS["C5"]
    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax, translation=translation)
    a_in = torch.from_numpy(fields.plane_wave_coefficients(pos, w.k, w.lmax).astype(np.complex64)).cuda()
    x = torch.zeros(w.N, w.nmax, dtype=torch.complex64, device="cuda")
    celes.celes_solve(ctx, a_in, x, restart=30, rtol=1e-4, max_iters=3)          # warm-up (allocations, caches)
    edge = [precond_edge, precond_edge, 0.0]
    pc = None
    if precond_edge > 0:
        celes.celes_precond_setup(ctx, edge)                                      # warm-up
    # three complete runs (set-up + solve each); the MEDIAN is reported and every run is listed.  The solve is
    # deterministic (same iterations every time) and repeats to 1 ms in isolation, but inside this script's full flow
    # about one preconditioned run in three has come out 15-70 ms slow for a reason not found
    runs = []
    for _ in range(3):
        x.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if precond_edge > 0:
            pc = celes.celes_precond_setup(ctx, edge)
            torch.cuda.synchronize()
        t_set = time.perf_counter() - t0
        info = celes.celes_solve(ctx, a_in, x, restart=30, rtol=1e-4, max_iters=2000, precond=pc is not None)
        torch.cuda.synchronize()
        runs.append((time.perf_counter() - t0, t_set, info))
    runs.sort(key=lambda r: r[0])
    sec, t_setup, info = runs[1]
    out = {"workload": f"C5: N={w.N} lmax={w.lmax} plane wave +z x-pol, GMRES(30), rtol 1e-4", "seconds": sec,
           "seconds_kind": "median of 3 complete runs (wall clock, set-up included)",
           "seconds_all": [r[0] for r in runs], "library_solve_seconds_all": [r[2]["seconds"] for r in runs],
           "iterations": info["iterations"], "matvecs": info["matvecs"], "rel_residual": info["rel_residual"],
           "converged": bool(all(r[2]["converged"] for r in runs))}
    if pc is not None:
        out["preconditioner"] = dict(pc, edge_nm=precond_edge, setup_seconds=t_setup,
                                     setup_note="replaces a warm-up set-up on the same context: device memory is reused, no "
                                                "allocator call; a context's first set-up adds its allocations (2-22 ms seen)",
                                     apply_roofline=precond_apply_roofline(celes, ctx, a_in, pc))
    return out, ctx, a_in


def main():
    args = parse()
    from paper_1706_02145_b200 import workloads
    w = workloads.CONFIGS[args.workload]
    if args.lmax:
        import dataclasses
        w = dataclasses.replace(w, name=f"{w.name}(lmax={args.lmax})", lmax=args.lmax)
    if args.impl == "reference":
        run_reference(args, w)
        return
    if args.solve:
        run_solve(args, w)
        return
    if args.far_field > 0:
        run_far_field(args, w)
        return
    if args.near_field > 0:
        run_near_field(args, w)
        return
    if args.gaussian_beam:
        run_gaussian_beam(args, w)
        return
    if args.shard == "receivers":
        run_sharded(args, w)
        return
    if args.cta_trace:
        run_cta_trace(args, w)
        return

    import torch
    import torch.distributed as dist
    import paper_1706_02145_b200 as celes
    from paper_1706_02145_b200 import fields, sass_count

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    pos, rad = workloads.positions(w)
    q = fields.mie_coefficients(w.lmax, w.k, rad, workloads.N_SPHERE)
    b_host = workloads.gaussian_coefficients(w.N, w.nmax, w.seed_b + rank)
    t0 = time.perf_counter()
    ctx = celes.celes_setup(pos, rad, q, w.k, w.lmax, translation=args.translation, hankel=args.hankel, levels=args.levels)
    setup_s = time.perf_counter() - t0
    cfg = celes.celes_launch_config(ctx)
    b = torch.from_numpy(b_host).cuda()
    y = torch.empty_like(b)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()
    pairs = w.N * (w.N - 1)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # FP32 peak of this GPU at its clocks of the moment (FFMA-only probes)
    probe = {v: celes.celes_fp32_peak_probe(v, 2048)["flops_per_s"] for v in (0, 1, 2, 3, 4)}
    for _ in range(args.warmup):
        celes.celes_coupling_matvec(ctx, b, y)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    step_ms = time_coupling(celes, ctx, b, y, args.steps, flush, stream)
    barrier()
    clocks = sampler.stop()
    total_ms = max_over_ranks(float(sum(step_ms)), world, "cuda")
    ms_per_step = total_ms / args.steps
    value = job_throughput(pairs, args.steps, world, total_ms)

    # end to end: pinned host buffers through the C ABI's host entry point, copies inside the timed region
    bh = torch.from_numpy(b_host).pin_memory()
    yh = torch.empty_like(bh).pin_memory()
    bh_np, yh_np = bh.numpy(), yh.numpy()
    celes.celes_coupling_matvec_host(ctx, bh_np, yh_np)
    barrier()
    t0 = time.perf_counter()
    for s in range(args.steps):
        celes.celes_coupling_matvec_host(ctx, bh_np, yh_np)
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, "cuda")
    e2e_value = job_throughput(pairs, args.steps, world, e2e_s * 1e3)

    if rank == 0:
        sm_count = torch.cuda.get_device_properties(local).multi_processor_count
        sm_max_mhz = clocks.get("sm_max_mhz") or measured_peaks().get("sm_max_mhz") or 1965.0
        sm_mhz = clocks.get("sm_mhz") or sm_max_mhz
        counts = sass_count.counts_for_bench(w.lmax, args.translation)
        roof = alu_roofline(counts, pairs, ms_per_step, sm_count, sm_max_mhz, sm_mhz)
        lane_rate = counts["lane_ops_per_pair"] * pairs / (ms_per_step * 1e-3)
        traffic = NCU_DRAM_BYTES_PER_LAUNCH.get((w.name, args.translation))
        roof.update({
            "traffic": None if traffic is None else traffic[0],
            "traffic_source": None if traffic is None else traffic[1],
            "translation": args.translation,
            "ffma_probe_tflops": {"reg": probe[0] / 1e12, "imm": probe[1] / 1e12, "f32x2": probe[2] / 1e12,
                                  "f32x2_3_register_operands": probe[3] / 1e12,
                                  "f32x2_shared_multiplicand": probe[4] / 1e12},
            "frac_of_ffma_probe": roof["achieved"] * 1e12 / max(probe.values()),
            "lane_rate_vs_3_operand_probe": lane_rate / (0.5 * probe[3]),
            "lane_rate_vs_shared_multiplicand_probe": lane_rate / (0.5 * probe[4])})
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"{w.name}: N={w.N} lmax={w.lmax} R=100nm n=1.52 lambda=550nm slab RSA ff=0.3",
                       "pairs_per_step": pairs, "l2": "flushed between timed iterations (256 MiB write)",
                       "launch": cfg, "hankel": args.hankel, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "setup_s": setup_s, "step_ms_min": float(min(step_ms)), "step_ms_median": float(np.median(step_ms))},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(b_host.nbytes),
                    "d2h_bytes_per_step": int(b_host.nbytes)},
            "gpu_launches": 3 * args.steps,
            "roofline": roof,
        }
        if w.name == "C4" and world == 1 and not args.lmax and not args.levels:
            # BASELINE.json's metric names N = 1e4 as well: the same measurement on C3, reported beside the headline
            w3 = workloads.CONFIGS["C3"]
            pos3, rad3 = workloads.positions(w3)
            ctx3 = celes.celes_setup(pos3, rad3, fields.mie_coefficients(w3.lmax, w3.k, rad3, workloads.N_SPHERE), w3.k,
                                     w3.lmax, translation=args.translation, hankel=args.hankel)
            b3 = torch.from_numpy(workloads.gaussian_coefficients(w3.N, w3.nmax, w3.seed_b)).cuda()
            y3 = torch.empty_like(b3)
            for _ in range(max(3, args.warmup)):
                celes.celes_coupling_matvec(ctx3, b3, y3)
            ms3 = float(np.median(time_coupling(celes, ctx3, b3, y3, 10, flush, stream)))
            p3 = w3.N * (w3.N - 1)
            r3 = alu_roofline(counts, p3, ms3, sm_count, sm_max_mhz, sm_mhz)
            line["also"] = {"workload": f"C3: N={w3.N} lmax={w3.lmax} (same recipe, 20 um slab)", "ms_per_step": ms3,
                            "value": p3 / (ms3 * 1e-3), "unit": UNIT, "steps": 10,
                            "launch": celes.celes_launch_config(ctx3),
                            "roofline": {k: r3[k] for k in ("frac", "fma_pipe_utilisation", "achieved", "peak", "unit")}}
            del ctx3
            # BASELINE.json config 5: the lmax = 4 kernel of the full solve, then the solve itself (time to solution and
            # iteration count), plain and with the paper's block-diagonal preconditioner
            solve, ctx5, a5 = solve_c5(celes, fields, workloads, args.translation)
            w5 = workloads.CONFIGS["C5"]
            b5 = torch.from_numpy(workloads.gaussian_coefficients(w5.N, w5.nmax, w5.seed_b)).cuda()
            y5 = torch.empty_like(b5)
            for _ in range(max(3, args.warmup)):
                celes.celes_coupling_matvec(ctx5, b5, y5)
            ms5 = float(np.median(time_coupling(celes, ctx5, b5, y5, 10, flush, stream)))
            p5 = w5.N * (w5.N - 1)
            c5 = sass_count.counts_for_bench(w5.lmax, args.translation)
            r5 = alu_roofline(c5, p5, ms5, sm_count, sm_max_mhz, sm_mhz)
            line["also_c5"] = {"workload": f"C5 geometry: N={w5.N} lmax={w5.lmax} (coupling matvec, L2 flushed)",
                               "ms_per_step": ms5, "value": p5 / (ms5 * 1e-3), "unit": UNIT, "steps": 10,
                               "launch": celes.celes_launch_config(ctx5), "roofline": r5}
            line["also_solve"] = solve
            del ctx5
            solve_pc, ctx5, _ = solve_c5(celes, fields, workloads, args.translation, precond_edge=PRECOND_EDGE_NM)
            line["also_solve_preconditioned"] = solve_pc
            del ctx5
        if not args.no_cpu_baseline and world == 1:
            rate, cores, n_recv, dt = oracle_sample_rate(w, pos, b_host, args.cpu_seconds)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{n_recv} seeded receivers x {w.N - 1} emitters ({dt:.1f} s)"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
