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
