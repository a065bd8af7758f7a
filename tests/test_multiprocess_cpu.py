"""N > 1 on CPU (gloo, world_size 2): the path does not shard (replicas only), so what there
is to cover is bench.py's plumbing -- the max-over-ranks reduction of the replicas' times and the reference arm
under torchrun (rank 0 alone runs and prints, the other ranks exit 0 without work)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
r = dist.get_rank()
got = bench.max_over_ranks(10.0 + 5.0 * r, dist, torch.device("cpu"))
assert got == 15.0, got
dist.barrier()
if r == 0:
    print("MAX_OK", got)
dist.destroy_process_group()
"""


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29653"] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_max_over_ranks_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    res = _torchrun([str(script)])
    assert res.returncode == 0, res.stderr[-2000:]
    assert "MAX_OK 15.0" in res.stdout


def test_reference_arm_under_torchrun_prints_one_line():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1",
                     "--ref-rows", "16"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
