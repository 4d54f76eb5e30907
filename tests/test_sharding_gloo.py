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


# ------------------------------------------------------------------- slab decomposition: plan, routing, transport ----
class _ToySlab:
    """CPU stand-in with the slab_* methods of binding.Ccake (tests of the HOST logic only: which message goes where and
    when).  Particles are (gid, x); a substep moves every owned particle by `drift`; ghosts are just recorded."""

    def __init__(self, gid, x, lo, hi, width, drift):
        self.gid, self.x = np.asarray(gid, dtype=np.int64), np.asarray(x, dtype=np.float64)
        self.lo, self.hi, self.w, self.drift = lo, hi, width, drift
        self.ghosts = {0: None, 1: None}
        self.arrivals = {0: None, 1: None}
        self.log = []

    def _pack(self, sel, buf):
        import torch
        n = int(sel.sum())
        buf[0, :n] = torch.as_tensor(self.x[sel])
        buf[28, :n] = torch.as_tensor(self.gid[sel].astype(np.float64))
        return n

    def slab_export_halo(self, side, k, buf):
        sel = (self.x < self.lo + self.w) if side == 0 else (self.x >= self.hi - self.w)
        self.log.append(("export_halo", side, k))
        return self._pack(sel, buf)

    def slab_import_ghosts(self, side, k, buf, count):
        self.log.append(("import_ghosts", side, k))
        self.ghosts[side] = (buf[28, :count].numpy().astype(np.int64).copy(), buf[0, :count].numpy().copy())

    def slab_substep(self, k):
        self.log.append(("substep", k))
        if k == 1:
            self.x = self.x + self.drift

    def slab_export_migrants(self, side, buf):
        sel = (self.x < self.lo) if side == 0 else (self.x >= self.hi)
        return self._pack(sel, buf)

    def slab_import_migrants(self, side, buf, count):
        self.arrivals[side] = (buf[28, :count].numpy().astype(np.int64).copy(), buf[0, :count].numpy().copy())

    def slab_commit(self):
        keep = (self.x >= self.lo) & (self.x < self.hi)
        gid, x = [self.gid[keep]], [self.x[keep]]
        for side in (0, 1):
            if self.arrivals[side] is not None:
                gid.append(self.arrivals[side][0]); x.append(self.arrivals[side][1])
        self.gid, self.x = np.concatenate(gid), np.concatenate(x)
        self.arrivals = {0: None, 1: None}
        return self.gid.size


def test_slab_plan():
    x = np.repeat(np.arange(31) * 0.1, 50)                  # 31 layers of 50 particles, as the eta slices of C4
    planes = sharding.slab_planes(x, 3)
    assert len(planes) == 2 and planes[0] < planes[1]
    assert all(not np.any(x == p) for p in planes)          # no particle on a plane
    counts = [int(np.sum((x >= sharding.slab_bounds(planes, k)[0]) & (x < sharding.slab_bounds(planes, k)[1]))) for k in range(3)]
    assert sum(counts) == x.size and max(counts) - min(counts) <= 50
    assert sharding.slab_bounds(planes, 0)[0] == -sharding.INF and sharding.slab_bounds(planes, 2)[1] == sharding.INF
    assert sharding.slab_halo_width(0.3, 0.05) == pytest.approx(1.3)
    assert [sharding.slab_owner(k, 4, 2) for k in range(4)] == [0, 0, 1, 1]
    with pytest.raises(ValueError):
        sharding.slab_planes(np.zeros(10), 2)


def _toy_event():
    rng = np.random.default_rng(11)
    x = np.sort(rng.uniform(0.0, 8.0, 400))
    return np.arange(400), x


def _slab_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        gid, x = _toy_event()
        K, width, drift = 4, 0.7, 0.3
        planes = sharding.slab_planes(x, K)
        local = {}
        for k in sharding.tile_range(K, rank, world):
            lo, hi = sharding.slab_bounds(planes, k)
            sel = (x >= lo) & (x < hi)
            local[k] = _ToySlab(gid[sel], x[sel], lo, hi, width, drift)
        drv = sharding.SlabDriver(local, K, 2, 400, lambda r, c: torch.zeros((r, c), dtype=torch.float64), rank=rank, world=world)
        drv.step(3)
        out = {k: (s.gid.tolist(), s.x.tolist(), {sd: (g[0].tolist() if g is not None else None) for sd, g in s.ghosts.items()}, s.log[:8])
               for k, s in local.items()}
        q.put((rank, out, drv.bytes_moved))
    finally:
        dist.destroy_process_group()


def test_slab_driver_world_size_2():
    """4 slabs on 2 ranks (2 each): one face between the ranks, one face inside each rank.  After 3 steps of a uniform drift
    every particle is owned by the slab its coordinate lies in, nothing is lost or doubled, and the ghosts of the last step
    are exactly the neighbours' particles within the halo width."""
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_slab_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    gid0, x0 = _toy_event()
    planes = sharding.slab_planes(x0, 4)
    slabs = {}
    for rank, out, moved in res:
        assert moved > 0
        slabs.update(out)
    assert sorted(slabs) == [0, 1, 2, 3]
    allgid = np.concatenate([np.array(slabs[k][0], dtype=np.int64) for k in range(4)])
    assert np.array_equal(np.sort(allgid), gid0)                      # a partition of the particles
    xend = x0 + 3 * 0.3
    for k in range(4):
        lo, hi = sharding.slab_bounds(planes, k)
        g = np.array(slabs[k][0], dtype=np.int64)
        assert np.allclose(np.array(slabs[k][1]), xend[g])
        assert np.all((xend[g] >= lo) & (xend[g] < hi))
        assert slabs[k][3][:3] == [("export_halo", 0, 0), ("export_halo", 1, 0), ("import_ghosts", 0, 0)] or k in (0, 3)
    # ghosts at the last step (state before its drift): the neighbours' particles within 0.7 of the shared face
    xlast = x0 + 2 * 0.3
    for k in range(4):
        lo, hi = sharding.slab_bounds(planes, k)
        if k > 0:
            want = gid0[(xlast < lo) & (xlast >= lo - 0.7) & (xlast >= sharding.slab_bounds(planes, k - 1)[0])]
            assert sorted(slabs[k][2][0]) == sorted(want.tolist())
        if k < 3:
            want = gid0[(xlast >= hi) & (xlast < hi + 0.7) & (xlast < sharding.slab_bounds(planes, k + 1)[1])]
            assert sorted(slabs[k][2][1]) == sorted(want.tolist())
