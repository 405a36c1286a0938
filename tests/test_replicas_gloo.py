"""The N>1 path of bench.py on CPU: world_size 2 over gloo.  Replicas only:
the exchange is max-over-ranks time and sum-over-ranks interactions, nothing on the data path."""
import importlib.util
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _load_replicas():
    # by path: importing the package would load libotoo.so, which this test does not need
    spec = importlib.util.spec_from_file_location("replicas", os.path.join(ROOT, "paper_1206_1199_b200", "replicas.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rep = _load_replicas()
    ms_local = [4.0, 5.5][rank]           # rank 1 is the slow one
    units_local = [7.0e9, 7.5e9][rank]
    ms, units = rep.aggregate(ms_local, units_local)
    val = rep.throughput(ms_local, units_local)
    dist.barrier()
    q.put((rank, ms, units, val, rep.replica_seed(1206, rank)))
    dist.destroy_process_group()


def test_replica_aggregation_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units, val, seed in res:
        assert ms == 5.5 and units == 14.5e9
        assert val == pytest.approx(14.5e9 / 5.5e-3)
        assert seed == 1206 + rank
    assert res[0][4] != res[1][4]


def test_aggregate_without_process_group():
    rep = _load_replicas()
    assert rep.aggregate(3.0, 10.0) == (3.0, 10.0)
    assert rep.throughput(2.0, 10.0) == pytest.approx(5000.0)


# ---- target sharding (PAPER III-E): partition logic and the combine step, on CPU
def _load_sharded():
    spec = importlib.util.spec_from_file_location("sharded", os.path.join(ROOT, "paper_1206_1199_b200", "sharded.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_group_ranges_partition_the_groups():
    import numpy as np
    sh = _load_sharded()
    for n, w in ((8192, 4), (10, 3), (3, 8), (0, 2), (131072, 8), (7, 1)):
        r = sh.group_ranges(n, w)
        assert len(r) == w and r[0][0] == 0 and sum(c for _, c in r) == n
        assert all(r[k][0] + r[k][1] == r[k + 1][0] for k in range(w - 1))          # contiguous, in key order
        assert max(c for _, c in r) - min(c for _, c in r) <= 1                        # the paper's N/P_GPU
    rng = np.random.default_rng(3)
    cost = rng.pareto(1.5, 5000) + 1.0                                                # a few very long lists
    r = sh.group_ranges(5000, 4, cost)
    assert r[0][0] == 0 and sum(c for _, c in r) == 5000 and all(r[k][0] + r[k][1] == r[k + 1][0] for k in range(3))
    shares = [cost[b:b + c].sum() for b, c in r]
    assert max(shares) <= cost.sum() / 4 + cost.max()                                 # balanced up to one group
    by_count = [cost[b:b + c].sum() for b, c in sh.group_ranges(5000, 4)]
    assert max(shares) <= max(by_count) * 1.0001
    assert sh.group_ranges(6, 3, np.zeros(6)) == sh.group_ranges(6, 3)
    assert sh.group_ranges(5000, 4, torch.from_numpy(cost)) == r                      # a tensor cost: same cuts


def _shard_worker(rank, world, port, q):
    import numpy as np
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sh = _load_sharded()
    n_groups, G = 37, 4
    n = n_groups * G - 1                                                               # ragged last group
    full = torch.arange(n * 4, dtype=torch.float32).reshape(-1, 4) + 1.0              # what one GPU would compute (sorted order)
    ok = True
    for cost in (None, np.linspace(1.0, 9.0, n_groups)):                               # equal counts; unequal, cost-balanced ranges
        ranges = sh.group_ranges(n_groups, world, cost)
        b, c = ranges[rank]
        rows = [(rb * G, min((rb + rc) * G, n)) for rb, rc in ranges]
        local = torch.full_like(full, -7.0)                                            # rows of the other ranks: ignored garbage
        local[rows[rank][0]:rows[rank][1]] = full[rows[rank][0]:rows[rank][1]]         # this rank's targets only
        ok = ok and bool(torch.equal(sh.gather_ranges(local, rows), full))
        lengths = torch.zeros(n_groups)
        lengths[b:b + c] = torch.arange(b, b + c, dtype=torch.float32) + 1.0           # per-group cost, zero outside the range
        ok = ok and bool(torch.equal(sh.combine(lengths), torch.arange(n_groups, dtype=torch.float32) + 1.0))
    b, c = sh.group_ranges(n_groups, world)[rank]
    q.put((rank, ok, (b, c)))
    dist.destroy_process_group()


def test_sharded_combine_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _ in res)
    assert res[0][2] == (0, 18) and res[1][2] == (18, 19)
