"""The N > 1 path of bench.py on CPU: replicas only, so the only cross-rank step is the
max-over-ranks of the device-timed seconds and the whole-job aggregation.  World size 2, gloo backend."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
t = bench.max_over_ranks(1.0 + rank, world)          # rank 1 is the slow one
v = bench.job_throughput(1000, 4, world, t)
if rank == 0:
    print(json.dumps({"t": t, "v": v, "world": world}))
dist.destroy_process_group()
"""


def test_job_throughput_is_all_ranks_over_the_slowest():
    import bench
    assert bench.max_over_ranks(0.5, 1) == 0.5
    assert bench.job_throughput(1000, 4, 1, 2.0) == 2000.0
    assert bench.job_throughput(1000, 4, 8, 2.0) == 16000.0


def test_two_ranks_gloo_take_the_maximum_time(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", "29617", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2 and d["t"] == 2.0 and d["v"] == 2 * 1000 * 4 / 2.0


def test_reference_arm_prints_the_contract_line():
    """bench.py --impl reference times the oracle on the host cores and prints one JSON line (bounded sample)."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["unit"] == "segments/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "c1"
