"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only).  The path has no
data-path collective; what the ranks share is the timing protocol -- barrier, slowest rank's time, whole-job
throughput = world x pairs / slowest time -- and the rule that only rank 0 of the reference arm works."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(code: str, nproc: int = 2, port: int = 29611):
    env = dict(os.environ, PYTHONPATH=ROOT)
    path = os.path.join(ROOT, ".pytest_cache", "multi_rank_snippet.py")      # torch.distributed.run wants a file
    os.makedirs(os.path.dirname(path), exist_ok=True)
    with open(path, "w") as f:
        f.write(code)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), path]
    return subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)


def test_slowest_rank_sets_the_job_throughput_gloo_world2():
    code = textwrap.dedent("""
        import json, os, sys
        import torch.distributed as dist
        sys.path.insert(0, os.environ["PYTHONPATH"])
        import bench
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        dist.barrier()
        mine = 100.0 + 50.0 * rank                       # rank 1 is the slow replica
        slowest = bench.max_over_ranks(mine, world, "cpu")
        value = bench.job_throughput(1000, 4, world, slowest)
        if rank == 0:
            print("RESULT " + json.dumps({"world": world, "slowest": slowest, "value": value}))
        dist.destroy_process_group()
    """)
    r = _torchrun(code)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RESULT ")]
    assert len(line) == 1                                # one line, from rank 0 only
    out = json.loads(line[0][7:])
    assert out["world"] == 2 and out["slowest"] == 150.0
    assert out["value"] == 2 * 1000 * 4 / 0.150


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1, "cpu") == 12.5
    assert bench.job_throughput(10, 2, 1, 1000.0) == 20.0


def test_row_slices_cover_and_balance():
    sys.path.insert(0, ROOT)
    from paper_1706_02145_b200 import sharding
    for N, world, align in ((10000, 8, 127), (100000, 3, 128), (50, 4, 50), (7, 2, 1), (5, 8, 1)):
        sl = sharding.row_slices(N, world, align)
        assert len(sl) == world and sl[0][0] == 0 and sl[-1][1] == N
        assert all(a[1] == b[0] for a, b in zip(sl[:-1], sl[1:])) and all(e >= s for s, e in sl)
        assert all(s % align == 0 for s, _ in sl)
        sizes = [e - s for s, e in sl]
        assert max(sizes) - min(sizes) <= align


def test_all_gather_of_row_shards_gloo_world2():
    """The one collective of the receiver-sharded mode: every rank contributes its rows of b (unequal
    counts) and ends up with the full vector, bit for bit, on both ranks."""
    code = textwrap.dedent("""
        import json, os, sys
        import numpy as np, torch
        import torch.distributed as dist
        sys.path.insert(0, os.environ["PYTHONPATH"])
        from paper_1706_02145_b200 import sharding, workloads
        dist.init_process_group("gloo")
        rank, world = dist.get_rank(), dist.get_world_size()
        N, nmax = 301, 30
        b = torch.from_numpy(workloads.gaussian_coefficients(N, nmax, 77))
        ok = True
        for align in (1, 128):
            slices = sharding.row_slices(N, world, align)
            r0, r1 = slices[rank]
            full = sharding.all_gather_rows(b[r0:r1].clone(), slices, rank)
            ok = ok and full.shape == b.shape and bool(torch.equal(torch.view_as_real(full), torch.view_as_real(b)))
        flags = [None] * world
        dist.all_gather_object(flags, ok)
        if rank == 0:
            print("RESULT " + json.dumps({"world": world, "ok": flags, "slices": sharding.row_slices(N, world, 128)}))
        dist.destroy_process_group()
    """)
    r = _torchrun(code, port=29613)
    assert r.returncode == 0, r.stderr[-2000:]
    out = json.loads([l for l in r.stdout.splitlines() if l.startswith("RESULT ")][0][7:])
    assert out["world"] == 2 and out["ok"] == [True, True]
    assert out["slices"] == [[0, 128], [128, 301]]


REFERENCE_KEYS = {"impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                  "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e", "gpu_launches"}


def _check_reference_line(line: dict, n_gpus: int):
    assert REFERENCE_KEYS <= set(line) and line["impl"] == "reference"
    assert line["metric"] == "sphere_pair_translations_per_s" and line["unit"] == "pairs/s" and line["higher_is_better"] is True
    assert line["n_gpus"] == n_gpus and line["steps"] == 1 and line["value"] > 0 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["cpu_baseline"]["value"] == line["value"] and "receivers" in line["cpu_baseline"]["sample"]
    assert line["e2e"] == {"value": line["value"], "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert "workload" in line["config"] and "model" not in line["config"]


def test_reference_arm_prints_the_contract_line_without_a_gpu():
    """bench.py --impl reference: the oracle, as it stands, on the host cores (the tier's reference arm); runs anywhere,
    prints exactly one JSON line with the arm's keys.  Config 1 (N = 50) keeps it to a second."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "C1",
                        "--steps", "1", "--warmup", "0"], cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    _check_reference_line(json.loads(lines[0]), 1)


def test_reference_arm_under_torchrun_only_rank0_works():
    """Launched like the GPU arm for N = 2 (torchrun, two ranks): rank 0 alone runs and prints, rank 1 exits 0 silently."""
    env = dict(os.environ, PYTHONPATH=ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", "29617", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1",
           "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, env=env, cwd=ROOT, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    _check_reference_line(json.loads(lines[0]), 2)
