"""N > 1 is "replicas only": no data-path collective, max-over-ranks timing, rank 0
reports the sum.  These tests run the rank plumbing of bench.py with world_size 2 on CPU (gloo)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(1.0 + rank, world, "cpu")          # ranks measured 1.0 and 2.0 ms
val = bench.aggregate_value(1000000, ms, world)
if rank == 0:
    print("RESULT", ms, val)
dist.destroy_process_group()
"""


def _torchrun(args, timeout=240):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29613"] + args
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_and_aggregate_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    r = _torchrun([str(w)])
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RESULT")]
    assert len(line) == 1                                   # only rank 0 reports
    _, ms, val = line[0].split()
    assert float(ms) == 2.0                                 # the slowest rank
    assert abs(float(val) - 2 * 1e6 / 2e-3 / 1e9) < 1e-12   # both ranks' bytes over that time


def test_reference_arm_under_torchrun_only_rank0_prints():
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
