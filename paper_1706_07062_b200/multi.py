"""Multi-GPU plumbing: geodesics are independent ("no need to consider inter-node
communication"), so N GPUs run N independent batches with no collective on the data path.  The only
cross-rank operations are the bookkeeping reductions below (time = max over ranks, work = sum)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_range(n_units: int, rank: int, world: int):
    """Contiguous [lo, hi) slice of n_units independent units (images, tiles, particles) for this rank;
    sizes differ by at most one and the slices tile [0, n_units) exactly."""
    base, extra = divmod(n_units, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def reduce_job(times, work, device="cpu"):
    """times: per-rank seconds (list) -> max over ranks; work: per-rank unit counts -> sum over ranks."""
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    w = torch.tensor(list(work), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return t.tolist(), w.tolist()
