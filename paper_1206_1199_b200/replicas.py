"""Multi-GPU plumbing of bench.py: replicas only.

north_star fixes one GPU and no partitioning of the path, so N GPUs run N independent replicas of the
workload (one process per GPU, different seeds) with no data-path collective.  The only exchange is
the timing contract: barrier, then the MAX of the per-rank step times and the SUM of the per-rank
interaction counts.  Works on any torch.distributed backend (nccl on the GPU box, gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def replica_seed(base_seed: int, rank: int) -> int:
    """every replica draws its own particles"""
    return int(base_seed) + int(rank)


def aggregate(ms_local: float, units_local: float, device: str = "cpu"):
    """(max over ranks of ms_local, sum over ranks of units_local); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(ms_local: float, units_local: float, device: str = "cpu") -> float:
    """whole-job units per second: all ranks' units over the slowest rank's time"""
    ms, units = aggregate(ms_local, units_local, device)
    return units / (ms * 1e-3)
