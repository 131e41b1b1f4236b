"""Host-side logic of the N>1 launch ("replicas only").

The path has no exchange step (BASELINE.json:north_star: "Everything runs on one GPU, with no
sharding, no collectives"), so with N ranks every rank runs an independent replica of the whole
hot path on its own GPU and its own random-vector seed.  The only communication is the timing
protocol of bench.py: a barrier on both sides of the timed region and the MAX over ranks of the
device time.  Backend-agnostic (nccl on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def world() -> tuple[int, int]:
    """(rank, world_size) of the initialised process group, or (0, 1)."""
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def replica_seed(seed: int, rank: int) -> int:
    """Seed of rank's replica: distinct random-phase streams per rank (the counter hash keys on
    (seed, r, i), so different seeds give independent vectors), rank 0 keeps the workload's."""
    return (int(seed) + 1000 * int(rank)) & (2**64 - 1)


def barrier(device: torch.device) -> None:
    if world()[1] > 1:
        dist.barrier()
    if device.type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(ms: float, device: torch.device) -> float:
    """MAX over ranks of a per-rank duration (every rank gets the result)."""
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    if world()[1] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, ms_max: float) -> float:
    """Units all ranks processed / the slowest rank's time (weak scaling: fixed work per rank)."""
    return units_per_rank * world()[1] / (ms_max * 1e-3)
