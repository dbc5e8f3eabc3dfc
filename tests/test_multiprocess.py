"""N > 1 host logic on CPU: world_size-2 gloo group.  The data path has no collective (tiles are
independent); what is distributed is the tile partition and the max-over-ranks
timing that bench.py reports."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2407_20469_b200.sharding import max_over_ranks, shard_tiles, sum_over_ranks


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_tiles, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = shard_tiles(n_tiles, rank, world)
        flags = torch.zeros(n_tiles, dtype=torch.int64)
        flags[list(mine)] = 1
        dist.all_reduce(flags)                                   # every tile owned exactly once
        t_max = max_over_ranks(10.0 + rank, dist)                # slowest rank decides the step time
        total = sum_over_ranks(len(mine), dist)
        q.put((rank, list(mine), flags.tolist(), t_max, total))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_tiles", [64, 7, 1])
def test_tile_partition_and_timing_over_two_ranks(n_tiles):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_tiles, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    owned = sum((g[1] for g in got), [])
    assert owned == list(range(n_tiles))                         # contiguous, ordered, complete
    for g in got:
        assert g[2] == [1] * n_tiles
        assert g[3] == 11.0 and g[4] == n_tiles
    assert abs(len(got[0][1]) - len(got[1][1])) <= 1


def test_shard_tiles_edges():
    assert list(shard_tiles(5, 0, 1)) == [0, 1, 2, 3, 4]
    assert [len(shard_tiles(20000, r, 8)) for r in range(8)] == [2500] * 8
    assert [len(shard_tiles(10, r, 4)) for r in range(4)] == [3, 3, 2, 2]
    assert len(shard_tiles(0, 1, 2)) == 0
    with pytest.raises(ValueError):
        shard_tiles(4, 2, 2)
    assert max_over_ranks(3.5) == 3.5
