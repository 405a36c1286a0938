"""Target sharding of one force calculation over several GPUs -- the paper's multi-device scheme.

PAPER.md III-E (L177-L185): "All OpenCL devices use the same tree data but each device only computes the
force for particles in a given range ... particles are sorted by their [space-filling-curve] keys so that we
divide the N particle into groups with N/P_GPU particles."  Here: every rank builds the same tree from the same
particles (a redundant 0.4-7 ms build instead of a broadcast), walks a contiguous range of target groups
(`group_begin`/`group_count` options of libotoo.so) and the ranks' outputs -- zero outside their range -- are
summed with one all-reduce (NCCL over NVLink on the GPU box, gloo in the CPU tests).  The paper names load
balance as the missing piece (L185); `group_ranges` can balance by a per-group cost (e.g. the previous
step's list lengths) instead of by count.

bench.py does NOT use this: BASELINE.json's north_star fixes one GPU and no partitioning (replicas only).
This module holds no force arithmetic; without a process group it degenerates to the single-GPU call.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def group_ranges(n_groups: int, world: int, cost=None):
    """Contiguous ranges [(begin, count)] * world covering 0..n_groups exactly once, in key order.
    cost=None: equal counts (the paper's N/P_GPU); else boundaries at equal shares of the summed cost."""
    n_groups, world = int(n_groups), int(world)
    if world < 1 or n_groups < 0:
        raise ValueError("world >= 1 and n_groups >= 0 required")
    if cost is None:
        cuts = [(n_groups * k) // world for k in range(world + 1)]
    else:
        c = np.asarray(cost, dtype=np.float64)
        if c.shape != (n_groups,) or (c < 0).any():
            raise ValueError("cost must be n_groups non-negative numbers")
        pre = np.concatenate([[0.0], np.cumsum(c)])
        tot = pre[-1]
        if tot <= 0:
            return group_ranges(n_groups, world)
        cuts = [0]
        for k in range(1, world):
            j = int(np.searchsorted(pre, tot * k / world, side="left"))
            cuts.append(min(max(j, cuts[-1]), n_groups))
        cuts.append(n_groups)
    return [(cuts[k], cuts[k + 1] - cuts[k]) for k in range(world)]


def combine(local: torch.Tensor) -> torch.Tensor:
    """Sum of the ranks' outputs (each zero outside its own range): one all-reduce; identity without a group."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(local, op=dist.ReduceOp.SUM)
    return local


class ShardedGravity:
    """otoo_gravity over `world` GPUs, one process per GPU; `otoo` is this rank's binding.Otoo."""

    def __init__(self, otoo, rank: int | None = None, world: int | None = None):
        on = dist.is_available() and dist.is_initialized()
        self.o = otoo
        self.rank = rank if rank is not None else (dist.get_rank() if on else 0)
        self.world = world if world is not None else (dist.get_world_size() if on else 1)
        self.cost = None          # per-group list lengths of the last call: balances the next one

    def gravity(self, pos_mass, n_crit, eps, theta, group_size, out=None):
        o = self.o
        o.otoo_build_tree(pos_mass, n_crit)                       # the same tree on every rank
        n_groups = (o.N + group_size - 1) // group_size
        cost = self.cost if (self.cost is not None and len(self.cost) == n_groups) else None
        begin, count = group_ranges(n_groups, self.world, cost)[self.rank]
        o.otoo_set_option("group_begin", begin)
        o.otoo_set_option("group_count", count)
        try:
            acc = o.otoo_gravity(eps, theta, group_size, out=out)
            nt, nc, npart = o.otoo_export_group_stats()
        finally:
            o.otoo_set_option("group_begin", 0)
            o.otoo_set_option("group_count", -1)
        lengths = torch.from_numpy((nc.astype(np.int64) + npart).astype(np.float32)).to(acc.device)
        self.cost = combine(lengths).cpu().numpy()                # every rank learns every group's cost
        return combine(acc)
