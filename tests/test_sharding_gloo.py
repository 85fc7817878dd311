"""World-size-2 gloo test of the N>1 host logic: independent units per rank, max-over-ranks timing, summed throughput."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1905_05515_b200.sharding import shard_units


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = shard_units(36, world, rank)
    t = torch.tensor([10.0 + rank], dtype=torch.float64)       # this rank's step time
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([float(len(mine))], dtype=torch.float64)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    g = [None] * world
    dist.all_gather_object(g, mine)
    q.put((rank, float(t.item()), float(n.item()), g))
    dist.destroy_process_group()


def test_two_ranks_partition_and_reduce():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    res = [q.get(timeout=120) for _ in ps]
    [p.join(timeout=60) for p in ps]
    for rank, tmax, n, g in res:
        assert tmax == 11.0 and n == 36.0
        assert sorted(g[0] + g[1]) == list(range(36)) and not set(g[0]) & set(g[1])
    assert shard_units(5, 8, 7) == [] and shard_units(5, 1, 0) == [0, 1, 2, 3, 4]
