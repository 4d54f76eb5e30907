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
