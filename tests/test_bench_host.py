"""Host-side logic of the N > 1 path, on CPU: whole-job aggregation (time = max over ranks,
units = sum over ranks) under torch.distributed/gloo with world_size 2, and the batch
sharding (members partitioned over ranks, no data-path collective)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    import workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)

    def rmax(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def rsum(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    # rank r "took" (10 + 5 r) ms for 1000 (r + 1) units
    value, t = bench.aggregate(10.0 + 5.0 * rank, 1000.0 * (rank + 1), world, rmax, rsum)
    # batch sharding: every member owned exactly once, parameters travel with the member
    p = W.config5(n=64, side=3, n_steps=1)
    mine = list(W.shard_members(p["batch"], rank, world))
    q = W.shard(p, rank, world)
    owned = torch.zeros(p["batch"], dtype=torch.float64)
    owned[mine] = 1.0
    dist.all_reduce(owned, op=dist.ReduceOp.SUM)
    ok = bool(torch.all(owned == 1.0)) and q["batch"] == len(mine) \
        and np.array_equal(q["delta"], np.asarray(p["delta"])[mine]) \
        and np.array_equal(q["sched_amp"], np.asarray(p["sched_amp"])[mine]) \
        and q["psi0"].shape == (len(mine), 64, 64)
    out.put((rank, value, t, ok, mine))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_and_sharding_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, t, ok, mine in res:
        assert t == 15.0                       # max over ranks
        assert value == pytest.approx(3000.0 / 15e-3)   # sum of units / max time
        assert ok
    assert res[0][4] == [0, 1, 2, 3, 4] and res[1][4] == [5, 6, 7, 8]


def test_aggregate_single_rank_identity():
    sys.path.insert(0, ROOT)
    import bench
    v, t = bench.aggregate(2.0, 100.0, 1)
    assert t == 2.0 and v == pytest.approx(100.0 / 2e-3)


@pytest.mark.parametrize("batch,world", [(64, 8), (9, 2), (3, 4), (0, 2), (7, 7)])
def test_shard_members_partition(batch, world):
    import workloads as W
    seen = []
    sizes = []
    for r in range(world):
        m = list(W.shard_members(batch, r, world))
        seen += m
        sizes.append(len(m))
    assert seen == list(range(batch))
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        W.shard_members(4, 4, 4)
