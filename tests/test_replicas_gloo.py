"""N>1 host logic on CPU: world_size-2 gloo run of the timing protocol bench.py uses
(barrier, MAX over ranks, whole-job value) and of the reference arm's rank gating."""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2509_06525_b200 import replicas

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dev = torch.device("cpu")
    assert replicas.world() == (rank, world)
    replicas.barrier(dev)
    ms = replicas.max_over_ranks(10.0 * (rank + 1), dev)          # rank 1 is the slow one
    value = replicas.whole_job_value(1.0e6, ms)
    with open(os.path.join(out, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "value": value, "seed": replicas.replica_seed(6525, rank)}, f)
    replicas.barrier(dev)
    dist.destroy_process_group()


def test_two_rank_gloo_timing_protocol(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    res = [json.load(open(tmp_path / f"r{r}.json")) for r in range(world)]
    assert res[0]["ms"] == res[1]["ms"] == 20.0                   # MAX over ranks, on every rank
    assert res[0]["value"] == res[1]["value"] == 2 * 1.0e6 / 20.0e-3
    assert res[0]["seed"] == 6525 and res[1]["seed"] == 7525      # distinct replicas


def test_single_process_defaults():
    assert replicas.world() == (0, 1)
    assert replicas.max_over_ranks(3.5, torch.device("cpu")) == 3.5
    assert replicas.whole_job_value(10.0, 1000.0) == 10.0
    assert replicas.replica_seed(2**64 - 1, 1) == 999


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--gpus", "2", "--steps", "1", "--warmup", "0"], env=env,
                       capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
