"""N > 1 path of bench.py on CPU (gloo, world_size 2).  The hot path does not shard in this build ("replicas
only"): the only cross-rank logic is the barrier, the MAX over ranks of the timed region and
the whole-job aggregate; the reference arm runs on rank 0 alone."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
dist.barrier()
ms = bench.max_over_ranks(ms_local, dist, "cpu")
val = bench.whole_job_value(world, 2.0e6, ms)
print(json.dumps({{"rank": rank, "ms": ms, "value": val}}))
dist.destroy_process_group()
"""


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["ms"] == 15.0                                  # the max, on every rank
        assert l["value"] == pytest.approx(2 * 2.0e6 / 15.0e-3 / 1e9)   # units of all ranks / max time


def test_reference_arm_runs_on_rank0_only_world2():
    r = _torchrun(["bench.py", "--gpus", "2", "--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                       # the other rank exits 0 without work
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
