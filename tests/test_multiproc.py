"""N > 1 is "replicas only": every rank runs the same independent step and the reported time is
the max over ranks.  This covers bench.py's rank plumbing (barrier, MAX all-reduce, whole-job aggregation, rank-0
printing, reference arm on rank 0 only) with world_size 2 on the gloo backend -- no GPU."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["PDLLM_ROOT"])
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# each replica "measures" a different time; the job time is the max over ranks, the job value aggregates replicas
ms = bench.max_over_ranks(10.0 * (rank + 1), world, device="cpu")
us = bench.replica_us_per_step(ms, steps=5, world=world)
dist.barrier()
if rank == 0:
    print(json.dumps({"ms": ms, "us": us, "world": world}))
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_replica_timing_is_max_over_ranks_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, PDLLM_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(script)]
    res = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["world"] == 2
    assert out["ms"] == pytest.approx(20.0)                  # max(10, 20)
    assert out["us"] == pytest.approx(1e3 * 20.0 / (5 * 2))  # world replicas of 5 steps ran in that time


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "tiny"], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0 and res.stdout.strip() == ""
    env["RANK"] = "0"
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--workload", "tiny"], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads(res.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "us"


def test_gpus_flag_without_one_rank_per_gpu_is_refused():
    """`bench.py --gpus 2` outside torchrun must not print an n_gpus=1 line: it exits non-zero (replicas need one rank per GPU)."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0",
                          "--workload", "tiny"], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode != 0 and res.stdout.strip() == "" and "one rank per GPU" in res.stderr
