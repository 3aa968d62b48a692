"""Multi-GPU plumbing: replicas only.  Environments are independent, so N ranks run N replicas of the
workload with no collective on the data path; the only cross-rank operations are a barrier around the
timed region and a MAX over ranks of the device-measured times."""
from __future__ import annotations

import torch
import torch.distributed as dist


def barrier(world: int) -> None:
    if world > 1:
        dist.barrier()
    if torch.cuda.is_available():
        torch.cuda.synchronize()


def max_over_ranks(values, world: int, device="cpu") -> list:
    """Element-wise MAX over ranks of a list of floats (identity when world == 1)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_rate(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Aggregate throughput: every rank processed `units_per_rank` units in at most `seconds_max`."""
    return world * units_per_rank / seconds_max


def rank_seed(base_seed: int, rank: int) -> int:
    """Replica r draws different trajectories (seed + r); replica 0 is the single-GPU workload."""
    return base_seed + rank
