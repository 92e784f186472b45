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


def shard_global_index(n: int, tile: int, rank: int, world: int) -> torch.Tensor:
    """Image ray index of every shard-local ray of `rank` when n rays are dealt out in tiles of `tile`
    consecutive indices, tile t to rank t mod world (gray2_init_null_shard):
    global = ((j // tile) * world + rank) * tile + j % tile, cut off at n (the last tile may be ragged)."""
    tiles = (n + tile - 1) // tile
    mine = torch.arange(rank, max(tiles, rank), world, dtype=torch.int64)          # this rank's tiles (may be none)
    idx = (mine[:, None] * tile + torch.arange(tile, dtype=torch.int64)[None, :]).reshape(-1)
    return idx[idx < n]


def gather_image(local: torch.Tensor, n: int, tile: int, world: int | None = None) -> torch.Tensor:
    """All ranks' shard-local arrays (last dimension = rays, in shard order) -> the array of the whole image
    in ray order, on every rank.  One all_gather of equal-sized padded pieces (NCCL on GPUs, gloo on CPU);
    with a single process it only undoes the tile permutation.  The integration itself never communicates."""
    if world is None:
        world = dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1
    counts = [int(shard_global_index(n, tile, r, world).numel()) for r in range(world)]
    longest = max(counts)
    lead = local.shape[:-1]
    padded = torch.zeros(lead + (longest,), dtype=local.dtype, device=local.device)
    padded[..., : local.shape[-1]] = local
    if world > 1:
        pieces = [torch.empty_like(padded) for _ in range(world)]
        dist.all_gather(pieces, padded)
    else:
        pieces = [padded]
    out = torch.empty(lead + (n,), dtype=local.dtype, device=local.device)
    for r in range(world):
        out[..., shard_global_index(n, tile, r, world).to(local.device)] = pieces[r][..., : counts[r]]
    return out


def reduce_job(times, work, device="cpu"):
    """times: per-rank seconds (list) -> max over ranks; work: per-rank unit counts -> sum over ranks."""
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    w = torch.tensor(list(work), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return t.tolist(), w.tolist()
