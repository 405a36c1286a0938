"""Target sharding of one force calculation over several GPUs -- the paper's multi-device scheme.

PAPER.md III-E (L177-L185): "All OpenCL devices use the same tree data but each device only computes the
force for particles in a given range ... particles are sorted by their [space-filling-curve] keys so that we
divide the N particle into groups with N/P_GPU particles."  Here: every rank builds the same tree from the same
particles (a redundant 0.4-6 ms build instead of a broadcast), walks a contiguous range of target groups
(`group_begin` / `group_count` options of libotoo.so) and writes its results in SORTED order (`output_sorted`),
where its targets are one contiguous run of rows.  The exchange is then an all-gather of those runs -- N/P x 16
bytes sent per rank, half of what an all-reduce of the zero-padded N x float4 moves -- and one `otoo_unsort`
back into the caller's order.  The paper names load balance as the missing piece (L185): the ranges can be cut
at equal shares of a per-group cost (the previous step's list lengths) instead of equal counts; the cost stays on
the device (one small all-reduce and a cumulative sum there, `world - 1` integers come to the host).

bench.py does NOT use this: BASELINE.json's north_star fixes one GPU and no partitioning (replicas only), and no
node with more than one GPU was available to this build: the path is covered by world_size-2 gloo tests on CPU
tensors (tests/test_replicas_gloo.py) and by a one-GPU test that runs the ranks' ranges one after the other.
This module holds no force arithmetic; without a process group it degenerates to the single-GPU call.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def group_ranges(n_groups: int, world: int, cost=None):
    """Contiguous ranges [(begin, count)] * world covering 0..n_groups exactly once, in key order.
    cost=None: equal counts (the paper's N/P_GPU); else boundaries at equal shares of the summed cost
    (a numpy array or a torch tensor on any device: the cumulative sum runs where the tensor lives)."""
    n_groups, world = int(n_groups), int(world)
    if world < 1 or n_groups < 0:
        raise ValueError("world >= 1 and n_groups >= 0 required")
    if cost is not None and not isinstance(cost, torch.Tensor):
        c = np.asarray(cost, dtype=np.float64)
        if c.shape != (n_groups,) or (c < 0).any():
            raise ValueError("cost must be n_groups non-negative numbers")
        cost = torch.from_numpy(c)
    if cost is not None and (cost.shape != (n_groups,) or bool((cost < 0).any())):
        raise ValueError("cost must be n_groups non-negative numbers")
    if cost is None or n_groups == 0 or float(cost.sum()) <= 0:
        cuts = [(n_groups * k) // world for k in range(world + 1)]
    else:
        pre = torch.cat([cost.new_zeros(1, dtype=torch.float64), torch.cumsum(cost.double(), 0)])
        marks = pre[-1] * torch.arange(1, world, dtype=torch.float64, device=pre.device) / world
        js = torch.searchsorted(pre, marks, right=False).tolist()          # world - 1 integers leave the device
        cuts = [0]
        for j in js:
            cuts.append(min(max(int(j), cuts[-1]), n_groups))
        cuts.append(n_groups)
    return [(cuts[k], cuts[k + 1] - cuts[k]) for k in range(world)]


def _on():
    return dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1


def gather_ranges(local_rows: torch.Tensor, row_ranges):
    """All-gather of the ranks' contiguous row ranges.  local_rows: (n, k) tensor whose rows [b, e) = row_ranges[rank]
    hold this rank's results (the others are ignored); returns the (n, k) tensor with every rank's rows in place.
    Ranges may differ in length (cost-balanced cuts): chunks are padded to the longest one."""
    if not _on():
        return local_rows
    rank, world = dist.get_rank(), dist.get_world_size()
    assert len(row_ranges) == world
    longest = max(e - b for b, e in row_ranges)
    b, e = row_ranges[rank]
    send = local_rows.new_zeros((longest,) + tuple(local_rows.shape[1:]))
    send[:e - b] = local_rows[b:e]
    recv = local_rows.new_empty((world * longest,) + tuple(local_rows.shape[1:]))
    dist.all_gather_into_tensor(recv, send)
    out = torch.empty_like(local_rows)
    for r, (rb, re) in enumerate(row_ranges):
        out[rb:re] = recv[r * longest:r * longest + (re - rb)]
    return out


def combine(local: torch.Tensor) -> torch.Tensor:
    """Sum of the ranks' tensors (each zero outside its own range): one all-reduce; identity without a group.
    Used for the small per-group cost vector; the N x float4 results go through gather_ranges."""
    if _on():
        dist.all_reduce(local, op=dist.ReduceOp.SUM)
    return local


class ShardedGravity:
    """otoo_gravity over `world` GPUs, one process per GPU; `otoo` is this rank's binding.Otoo."""

    def __init__(self, otoo, rank: int | None = None, world: int | None = None):
        on = dist.is_available() and dist.is_initialized()
        self.o = otoo
        self.rank = rank if rank is not None else (dist.get_rank() if on else 0)
        self.world = world if world is not None else (dist.get_world_size() if on else 1)
        self.cost = None          # per-group list lengths of the last call (device tensor): balances the next one

    def gravity(self, pos_mass, n_crit, eps, theta, group_size, out=None):
        o = self.o
        o.otoo_build_tree(pos_mass, n_crit)                       # the same tree on every rank
        n_groups = (o.N + group_size - 1) // group_size
        cost = self.cost if (self.cost is not None and self.cost.shape[0] == n_groups) else None
        ranges = group_ranges(n_groups, self.world, cost)
        begin, count = ranges[self.rank]
        o.otoo_set_option("group_begin", begin)
        o.otoo_set_option("group_count", count)
        o.otoo_set_option("output_sorted", 1)
        try:
            rows = o.otoo_gravity(eps, theta, group_size)         # sorted order: this rank's targets are rows [b G, e G)
            _, nc, npart = o.otoo_export_group_stats(on_device=True)
        finally:
            o.otoo_set_option("group_begin", 0)
            o.otoo_set_option("group_count", -1)
            o.otoo_set_option("output_sorted", 0)
        self.cost = combine((nc + npart).to(torch.float32))       # zero outside the range: the sum is every group's cost
        row_ranges = [(b * group_size, min((b + c) * group_size, o.N)) for b, c in ranges]
        return o.otoo_unsort(gather_ranges(rows, row_ranges), out=out)
