"""world_size-2 gloo test (CPU) of the N > 1 host logic: disjoint frame shards, max-over-ranks timing, aggregate rate.
The data path has no collective (frames are independent), so this is all there is to the multi-GPU plumbing."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1712_06913_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_grids, out):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = shard.shard_range(n_grids, rank, world)
        mine = torch.zeros(n_grids, dtype=torch.int64)
        mine[a:b] = 1
        dist.all_reduce(mine)                                   # test-only collective: coverage of the shards
        ms = shard.max_over_ranks(10.0 + 5.0 * rank, dist)       # rank 1 is the slow one
        seeds = list(shard.frame_seeds(rank, 3))
        gathered = [None] * world
        dist.all_gather_object(gathered, seeds)
        if rank == 0:
            out.put((mine.tolist(), ms, gathered))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_cover_all_grids_once_and_time_is_the_slowest_ranks():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port, world, n_grids = _free_port(), 2, 7
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_grids, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    cover, ms, seeds = out.get()
    assert cover == [1] * n_grids                               # every grid imaged by exactly one rank
    assert ms == 15.0                                           # MAX over ranks
    assert seeds == [[0, 1, 2], [3, 4, 5]]                      # weak scaling: disjoint frames per rank
    assert shard.aggregate_rate(100, world, ms) == pytest.approx(200 / 0.015)


@pytest.mark.parametrize("n,world", [(0, 3), (1, 4), (7, 2), (32000, 8), (5, 5)])
def test_shard_range_partitions(n, world):
    parts = [shard.shard_range(n, r, world) for r in range(world)]
    assert parts[0][0] == 0 and parts[-1][1] == n
    assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
    sizes = [b - a for a, b in parts]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(n, world, world)
