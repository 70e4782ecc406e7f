"""World-size-2 gloo test (CPU) of the N>1 host logic: CCD sharding, barrier, max-over-ranks timing."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_08593_b200 import shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = shard.shard_ccds(60, rank, world)
    gathered = [None] * world
    dist.all_gather_object(gathered, mine)
    dist.barrier()
    ms = shard.max_over_ranks(10.0 + 5.0 * rank)
    q.put((rank, mine, gathered, ms, shard.aggregate_rate(len(mine), world, ms)))
    dist.destroy_process_group()


def test_shard_partition_is_exact():
    for world in (1, 2, 3, 8):
        parts = [shard.shard_ccds(60, r, world) for r in range(world)]
        allc = sorted(c for p in parts for c in p)
        assert allc == list(range(60))
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_world2_gloo_max_over_ranks_and_sharding():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mine, gathered, ms, rate in res:
        assert ms == 15.0                      # max over ranks, not the local time
        assert sorted(gathered[0] + gathered[1]) == list(range(60))
        assert set(gathered[0]).isdisjoint(gathered[1])
        assert abs(rate - 2 * 30 / 15e-3) < 1e-6
