"""World-size-2 gloo test (CPU) of bench.py's multi-rank host logic: per-rank seeds differ, times are reduced with
MAX over ranks, the job value is the weak-scaling aggregate, and only rank 0 of the reference arm reports."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
ms, e2e = bench.max_over_ranks([10.0 + rank, 3.0 - rank], world, torch.device("cpu"))
val = bench.whole_job_value(1000, world, ms)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "e2e": e2e, "value": val}))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_weak_scaling_value_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29653", str(script)],
                         capture_output=True, text=True, timeout=240, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    import json

    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["ms"] == 11.0 and r["e2e"] == 3.0  # MAX over ranks of (10, 11) and (3, 2)
    assert r["value"] == pytest.approx(2 * 1000 / 11e-3)


def test_reference_arm_only_rank0_reports():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
