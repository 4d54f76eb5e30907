"""Multi-process CPU test (gloo, world_size 2) of the N > 1 host logic: tile sharding, max-over-ranks timing and
the reduction of conserved totals.  The data path itself has no collective (DESIGN.md §"Multi-GPU")."""
import os
import socket

import numpy as np
import pytest

from paper_2511_22852_b200 import sharding


def test_tile_range_partitions_exactly():
    for n in (0, 1, 7, 10, 13):
        for world in (1, 2, 3, 4, 8):
            got = [t for r in range(world) for t in sharding.tile_range(n, r, world)]
            assert got == list(range(n))
            sizes = [len(sharding.tile_range(n, r, world)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.tile_range(4, 2, 2)


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        tiles = list(sharding.tile_range(5, rank, world))
        tmax = sharding.reduce_max(10.0 + rank)
        tot = np.zeros(16)
        tot[0] = 1.5
        tot[1] = 100.0 * (rank + 1)
        tot[5] = float(len(tiles))
        tot[12] = 0.25 * (rank + 1)
        red = sharding.reduce_totals(tot)
        q.put((rank, tiles, tmax, red.tolist()))
    finally:
        dist.destroy_process_group()


def test_reductions_world_size_2():
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 1, 2] and res[1][1] == [3, 4]
    for r in res:
        assert r[2] == 11.0
        red = np.array(r[3])
        assert red[0] == 1.5 and red[1] == 300.0 and red[5] == 5.0 and red[12] == 0.5


def test_reductions_are_identity_without_a_group():
    assert sharding.reduce_max(3.0) == 3.0
    assert np.array_equal(sharding.reduce_totals(np.arange(16.0)), np.arange(16.0))
