"""Multi-GPU is "replicas only": no data-path collective, the only exchange
is the max-over-ranks of the device time.  world_size-2 gloo runs of that host logic on CPU, and of
the reference arm's "rank 0 alone prints" rule under torchrun."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["PFC_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
t = bench.max_over_ranks(0.5 + rank)            # rank r "measured" 0.5 + r seconds
v = bench.job_value(1000, 10, world, t)
dist.barrier()
if rank == 0:
    print(json.dumps({"t": t, "value": v, "world": world}))
dist.destroy_process_group()
"""


def _torchrun(args, env=None):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29611"] + args
    e = dict(os.environ, PFC_ROOT=ROOT, OMP_NUM_THREADS="2")
    e.update(env or {})
    return subprocess.run(cmd, cwd=ROOT, env=e, capture_output=True, text=True, timeout=600)


def test_max_over_ranks_and_job_value_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["world"] == 2 and out["t"] == 1.5               # the slower rank
    assert out["value"] == pytest.approx(2 * 1000 * 10 / 1.5)  # both replicas' atoms count


def test_reference_arm_prints_once_under_torchrun():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--config", "0", "--steps", "2",
                   "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["cpu_baseline"]["kind"] == "oracle"
    assert out["e2e"]["h2d_bytes_per_step"] == 0 and out["value"] > 0
