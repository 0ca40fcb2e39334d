"""Host logic of bench.py's N > 1 path (replicas only) on CPU: world_size 2 over gloo.
Each rank draws its own catalog (seed 2 + rank), the elapsed time is the MAX over ranks, the value is
the whole-job aggregate, and the reference arm runs on rank 0 alone."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import numpy as np
import torch, torch.distributed as dist
import bench
rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
class A: objects = 6; freqs = 64
cat = bench.make_catalog(A, rank)
elapsed = 100.0 * (rank + 1)                      # rank 1 is the slow one
dist.barrier()
m = bench.max_over_ranks(elapsed, dist, torch.device("cpu"))
v = bench.job_throughput(world, cat.n_objects * cat.n_freq, 3, m)
sums = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
dist.all_gather(sums, torch.tensor([float(cat.times.sum())], dtype=torch.float64))
print(json.dumps({"rank": rank, "max_ms": m, "value": v, "sums": [float(s) for s in sums]}), flush=True)
dist.destroy_process_group()
"""


def _env(rank, world, port):
    e = dict(os.environ)
    e.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
             MASTER_PORT=str(port))
    return e


def test_two_rank_timing_and_aggregation_over_gloo():
    port = 29500 + os.getpid() % 500
    procs = [subprocess.Popen([sys.executable, "-c", WORKER, ROOT], env=_env(r, 2, port), stdout=subprocess.PIPE,
                              stderr=subprocess.PIPE, text=True) for r in range(2)]
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["max_ms"] == 200.0                               # MAX over ranks, on every rank
        assert abs(o["value"] - 2 * 6 * 64 * 3 / 0.2) < 1e-6      # whole-job aggregate
        assert o["sums"][0] != o["sums"][1]                       # each rank has its own catalog (seed 2 + rank)


def test_reference_arm_runs_on_rank_zero_only():
    """bench.py --impl reference under torchrun's environment: rank 1 exits 0 without output or work."""
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=_env(1, 2, 29999), capture_output=True, text=True,
                       timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""
