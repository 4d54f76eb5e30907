"""Host-side logic of the multi-GPU path (DESIGN.md §"Multi-GPU"): the hot path shards by independent event tiles
— one process per GPU, each rank evolves its own tiles, no data-path collective.  The only exchanges are the timing
reduction (max over ranks) and the sum of the conserved totals; both go through torch.distributed (NCCL on GPUs,
gloo in the CPU tests)."""
from __future__ import annotations

import numpy as np


def tile_range(n_tiles: int, rank: int, world: int) -> range:
    """Contiguous, balanced split of n_tiles independent event tiles: the first (n_tiles % world) ranks get one more."""
    if world <= 0 or not (0 <= rank < world) or n_tiles < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_tiles, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def _tensor(x, device):
    import torch
    return torch.as_tensor(np.asarray(x, dtype=np.float64), device=device)


def reduce_max(value: float, device="cpu") -> float:
    """max over ranks of a device time; identity without an initialised process group."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = _tensor([value], device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_totals(totals, device="cpu") -> np.ndarray:
    """Job-wide conserved totals from per-rank ccake_conserved_totals vectors: additive entries (E, P_i, S, N_q,
    sum m, work, counts) are summed, x0 and max|trace pi| take the max."""
    import torch.distributed as dist
    t = np.asarray(totals, dtype=np.float64).copy()
    if not (dist.is_available() and dist.is_initialized()):
        return t
    add = _tensor(t, device)
    mx = add.clone()
    dist.all_reduce(add, op=dist.ReduceOp.SUM)
    dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    out = add.cpu().numpy()
    for k in (0, 12):
        out[k] = float(mx[k].item())
    return out


# ------------------------------------------------------------------------------------------------------------------
# Slab decomposition of ONE event (include/ccake.h "Slab decomposition"): host logic and transport.
# The selection, packing and unpacking of the messages run in the library's kernels (csrc/slab.cuh); what lives here is
# the plan (where to cut), the order of the calls, and moving the message buffers: a hand-over inside one process, or
# torch.distributed send / recv (NCCL between GPUs, gloo in the CPU tests).
SLAB_ROWS = 29          # 28 state fields + the global particle id
SLAB_REC_ROWS = 32      # a gradient record (narrow halos): the payload columns of the gradient pass and the position
INF = 1.0e300


def slab_planes(coord, n_slabs: int):
    """Cut planes along one coordinate so that the slabs hold (nearly) equal numbers of particles: n_slabs - 1 increasing
    values, each halfway between two neighbouring distinct coordinate values (no particle sits on a plane)."""
    x = np.sort(np.asarray(coord, dtype=np.float64))
    if n_slabs < 1 or x.size < n_slabs:
        raise ValueError("bad slab arguments")
    planes = []
    for k in range(1, n_slabs):
        i = (k * x.size) // n_slabs
        j = i
        while j < x.size and x[j] == x[i - 1]:          # move up to the next distinct value
            j += 1
        if j >= x.size:
            raise ValueError("cannot cut: too many particles share one coordinate value")
        planes.append(0.5 * (x[i - 1] + x[j]))
    if any(b <= a for a, b in zip(planes, planes[1:])):
        raise ValueError("cut planes are not increasing")
    return planes


def slab_bounds(planes, k: int):
    """[lo, hi) of slab k for the planes of slab_planes (the outer slabs are open-ended)."""
    lo = -INF if k == 0 else planes[k - 1]
    hi = INF if k == len(planes) else planes[k]
    return lo, hi


def slab_halo_width(h: float, dx0: float, narrow: bool = False) -> float:
    """Wide halos: two kernel supports (the smoothing sums of the neighbours of an owned particle are recomputed on ghosts)
    plus the drift of the particles on both sides during one step (|v| < 1).  Narrow halos: one kernel support plus the
    drift; the gradient records of the ghosts then come from their owners in a second message per substep."""
    return (2.0 if narrow else 4.0) * h + 2.0 * dx0


def slab_owner(k: int, n_slabs: int, world: int) -> int:
    """Rank that holds slab k: contiguous blocks of slabs per rank, as tile_range."""
    for r in range(world):
        if k in tile_range(n_slabs, r, world):
            return r
    raise ValueError("slab index out of range")


class SlabDriver:
    """Runs RK steps of one event decomposed into n_slabs slabs.  `local` maps the global index of every slab this rank
    holds to an object with the slab_* methods of binding.Ccake; buffers are made by `new_buffer(rows, cap)` (a torch
    tensor on the right device).  Neighbouring slabs on the same rank hand their messages over directly; slabs on other
    ranks are reached with torch.distributed point-to-point calls, all messages of a phase posted together."""

    def __init__(self, local: dict, n_slabs: int, nsub: int, buf_cap: int, new_buffer, rank: int = 0, world: int = 1,
                 narrow: bool = False):
        self.local, self.K, self.nsub, self.cap = dict(local), int(n_slabs), int(nsub), int(buf_cap)
        self.rank, self.world = rank, world
        self.new_buffer = new_buffer
        self.narrow = bool(narrow)          # the contexts were loaded with slab_halo_width(..., narrow=True)
        self.rows = SLAB_REC_ROWS if narrow else SLAB_ROWS        # one buffer size serves both kinds of message
        self.send = {k: [new_buffer(self.rows, buf_cap), new_buffer(self.rows, buf_cap)] for k in self.local}
        self.recv = {k: [new_buffer(self.rows, buf_cap), new_buffer(self.rows, buf_cap)] for k in self.local}
        self.bytes_moved = 0

    def _neighbour(self, k, side):
        nb = k - 1 if side == 0 else k + 1
        return nb if 0 <= nb < self.K else None

    def _exchange(self, export, accept, rows=SLAB_ROWS):
        """One phase: every local slab exports towards both faces, the messages travel, every local slab accepts what
        arrived at its faces (low face first).  export(k, side, buf) -> count; accept(k, side, buf, count).  rows = rows of
        a message that carry data (the buffers may have more)."""
        import torch
        arrived = {}                      # (slab, side) -> (buffer, count)
        remote = []                       # (dst rank, dst slab, dst side, buffer, count)
        for k in sorted(self.local):
            for side in (0, 1):
                nb = self._neighbour(k, side)
                if nb is None:
                    continue
                cnt = export(k, side, self.send[k][side])
                if cnt > self.cap:
                    raise RuntimeError("slab message exceeds the buffer capacity")
                self.bytes_moved += 8 * rows * cnt
                if nb in self.local:
                    arrived[(nb, 1 - side)] = (self.send[k][side], cnt)
                else:
                    remote.append((slab_owner(nb, self.K, self.world), nb, 1 - side, self.send[k][side], cnt))
        if self.world > 1:
            import torch.distributed as dist
            # what this rank expects: one message per (local slab, face) whose neighbour lives elsewhere
            expect = [(slab_owner(self._neighbour(k, side), self.K, self.world), k, side) for k in sorted(self.local) for side in (0, 1)
                      if self._neighbour(k, side) is not None and self._neighbour(k, side) not in self.local]
            dev = self.send[next(iter(self.local))][0].device
            scnt = [torch.tensor([c], dtype=torch.int64, device=dev) for (_, _, _, _, c) in remote]
            rcnt = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in expect]
            ops = [dist.P2POp(dist.isend, t, r[0], tag=2 * r[1] + r[2]) for t, r in zip(scnt, remote)]
            ops += [dist.P2POp(dist.irecv, t, e[0], tag=2 * e[1] + e[2]) for t, e in zip(rcnt, expect)]
            if ops:
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
            counts = [int(t.item()) for t in rcnt]
            sdat = [b[:rows, :c].contiguous() for (_, _, _, b, c) in remote]
            rdat = [self.new_buffer(rows, max(c, 1))[:, :c].contiguous() for c in counts]
            ops = [dist.P2POp(dist.isend, t, r[0], tag=2 * r[1] + r[2]) for t, r in zip(sdat, remote) if t.numel()]
            ops += [dist.P2POp(dist.irecv, t, e[0], tag=2 * e[1] + e[2]) for t, e in zip(rdat, expect) if t.numel()]
            if ops:
                for w in dist.batch_isend_irecv(ops):
                    w.wait()
            for (src, k, side), t, c in zip(expect, rdat, counts):
                if c > self.cap:
                    raise RuntimeError("slab message exceeds the buffer capacity")
                self.recv[k][side][:rows, :c] = t
                arrived[(k, side)] = (self.recv[k][side], c)
        elif remote:
            raise RuntimeError("a neighbouring slab is not local and there is no process group")
        for k in sorted(self.local):
            for side in (0, 1):
                if (k, side) in arrived:
                    buf, cnt = arrived[(k, side)]
                    accept(k, side, buf, cnt)

    def refresh_ghosts(self):
        """Halo exchange at the current state, so that derived fields and conserved totals of the owned particles near
        the faces see complete neighbours (ccake_read_fields / ccake_conserved_totals evaluate at the current state)."""
        self.drop_ghosts()
        self._exchange(lambda k, side, buf: self.local[k].slab_export_halo(side, 0, buf),
                       lambda k, side, buf, cnt: self.local[k].slab_import_ghosts(side, 0, buf, cnt))
        self.ghosts_present = True

    def drop_ghosts(self):
        if getattr(self, "ghosts_present", False):
            for k in sorted(self.local):
                self.local[k].slab_commit()          # nothing migrates at an unchanged state: the ghosts go, the owned stay
            self.ghosts_present = False

    def step(self, nsteps: int = 1):
        self.drop_ghosts()
        for _ in range(nsteps):
            for s in range(self.nsub):
                self._exchange(lambda k, side, buf: self.local[k].slab_export_halo(side, s, buf),
                               lambda k, side, buf, cnt: self.local[k].slab_import_ghosts(side, s, buf, cnt))
                if self.narrow:
                    for k in sorted(self.local):
                        self.local[k].slab_substep_part(s, 1)                      # a1-a5
                    self._exchange(lambda k, side, buf: self.local[k].slab_export_records(side, buf),
                                   lambda k, side, buf, cnt: self.local[k].slab_import_records(side, buf, cnt), rows=SLAB_REC_ROWS)
                    for k in sorted(self.local):
                        self.local[k].slab_substep_part(s, 2)                      # a6-a8
                else:
                    for k in sorted(self.local):
                        self.local[k].slab_substep(s)
            self._exchange(lambda k, side, buf: self.local[k].slab_export_migrants(side, buf),
                           lambda k, side, buf, cnt: self.local[k].slab_import_migrants(side, buf, cnt))
            for k in sorted(self.local):
                self.local[k].slab_commit()
