"""World-size-2 gloo test of the multi-GPU host logic: slices are sharded
over ranks with no data-path collective; only the timing (max over ranks) and the bookkeeping
cross ranks.  Runs on CPU."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2601_12378_b200 import shard_slices


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_slices, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    first, count = shard_slices(n_slices, rank, world)
    mine = torch.zeros(n_slices, dtype=torch.int64)
    mine[first:first + count] = 1
    dist.all_reduce(mine)                                   # every slice owned exactly once
    t = torch.tensor([10.0 + rank], dtype=torch.float64)    # per-rank elapsed ms -> max over ranks
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    q.put((rank, first, count, mine.tolist(), float(t.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_cover_and_max_timing_world2():
    world, n = 2, 513
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = [q.get(timeout=120) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, first, count, cover, tmax in res:
        assert cover == [1] * n
        assert tmax == 11.0
    res.sort()
    assert res[0][1] == 0 and res[0][2] == 257 and res[1][1] == 257 and res[1][2] == 256


def test_shard_slices_edge_cases():
    assert shard_slices(0, 0, 4) == (0, 0)
    assert [shard_slices(3, r, 4) for r in range(4)] == [(0, 1), (1, 1), (2, 1), (3, 0)]
    tot = sum(shard_slices(1000, r, 8)[1] for r in range(8))
    assert tot == 1000
