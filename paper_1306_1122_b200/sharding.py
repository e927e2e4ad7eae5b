"""Point sharding across ranks.

Every field point is independent ("pointwise method"; PAPER.md:143, 161 name
MPI + CUDA over the points as the next step), so the multi-GPU path partitions the POINTS, replicates
the boundary (<= 34 MB) and has no data-path collective inside eval / solve.  This module is host
logic only (index arithmetic and torch.distributed plumbing); it holds none of the method's
arithmetic and works with any backend (nccl on GPUs, gloo in the CPU tests).

    idx  = shard_indices(M, rank, world, mode)     # this rank's point ids
    ...    run dbie_eval / dbie_solve on x[idx], y[idx], z[idx]
    full = gather_points(dist, local, M, mode)     # optional: every rank gets all M results
    ms, work = reduce_over_ranks(dist, device, ms, work)   # timing: max, work: sum
"""
from __future__ import annotations

import numpy as np

MODES = ("contiguous", "interleaved")


def shard_bounds(M: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slab [lo, hi) of rank `rank`: sizes differ by at most one point."""
    if M < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad shard request M={M} rank={rank} world={world}")
    base, extra = divmod(M, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_indices(M: int, rank: int, world: int, mode: str = "contiguous") -> np.ndarray:
    """Point ids owned by `rank`.  "contiguous": a slab (keeps z-layers together); "interleaved":
    every world-th point, which evens out the per-point iteration counts of the lambda search
    (neighbouring points converge after similar numbers of iterations)."""
    if mode not in MODES:
        raise ValueError(f"mode must be one of {MODES}")
    if mode == "contiguous":
        lo, hi = shard_bounds(M, rank, world)
        return np.arange(lo, hi, dtype=np.int64)
    if M < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"bad shard request M={M} rank={rank} world={world}")
    return np.arange(rank, M, world, dtype=np.int64)


def shard_sizes(M: int, world: int, mode: str = "contiguous") -> list[int]:
    return [int(shard_indices(M, r, world, mode).size) for r in range(world)]


def _world(dist) -> int:
    return dist.get_world_size() if (dist is not None and dist.is_initialized()) else 1


def broadcast_boundary(dist, bx, by, bz, src: int = 0):
    """Replicate the boundary from rank `src` (in place; tensors on the backend's device)."""
    if _world(dist) > 1:
        for t in (bx, by, bz):
            dist.broadcast(t, src=src)
    return bx, by, bz


def gather_points(dist, local, M: int, mode: str = "contiguous"):
    """All-gather per-point results.  `local`: tensor [..., m_rank] whose last axis runs over this
    rank's points in shard order.  Returns [..., M] in global point order on every rank."""
    import torch
    world = _world(dist)
    if world == 1:
        return local
    rank = dist.get_rank()
    sizes = shard_sizes(M, world, mode)
    if local.shape[-1] != sizes[rank]:
        raise ValueError(f"rank {rank} holds {local.shape[-1]} points, expected {sizes[rank]}")
    mmax = max(sizes)
    pad = torch.zeros(local.shape[:-1] + (mmax,), dtype=local.dtype, device=local.device)
    pad[..., : sizes[rank]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad.contiguous())
    full = torch.empty(local.shape[:-1] + (M,), dtype=local.dtype, device=local.device)
    for r in range(world):
        idx = torch.from_numpy(shard_indices(M, r, world, mode)).to(local.device)
        full[..., idx] = parts[r][..., : sizes[r]]
    return full


def reduce_over_ranks(dist, device, ms: float, work: float) -> tuple[float, float]:
    """The bench contract's aggregate: max over ranks of the device time, sum of the work."""
    import torch
    if _world(dist) == 1:
        return ms, work
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    w = torch.tensor([work], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return float(t.item()), float(w.item())
