"""N > 1 on CPU (gloo, world_size 2): the path does not shard ("replicas only"), so what there is to
cover is the launch contract of bench.py under torchrun and its one scalar reduction (max over ranks)."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(args, port):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=600)


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"], 29731)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, res.stdout
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["n_gpus"] == 2 and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["e2e"]["h2d_bytes_per_step"] == 0


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
t = bench.max_over_ranks(1.0 + rank)            # rank r took 1 + r seconds
v = bench.aggregate_value(1e9, t, world)        # each replica did 1e9 points
dist.barrier()
if rank == 0:
    print("RESULT %%d %%.6f %%.6f" %% (world, t, v))
dist.destroy_process_group()
"""


def test_max_over_ranks_and_weak_scaling_aggregate_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    res = _torchrun([str(script)], 29732)
    assert res.returncode == 0, res.stderr[-2000:]
    out = [ln for ln in res.stdout.splitlines() if ln.startswith("RESULT")]
    assert len(out) == 1
    _, world, t, v = out[0].split()
    assert int(world) == 2
    assert float(t) == pytest.approx(2.0)       # the slowest rank
    assert float(v) == pytest.approx(1.0)       # 2 replicas x 1e9 points / 2 s = 1 Gpts/s
