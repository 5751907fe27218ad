"""Host-side sharding of independent events across ranks.

The path partitions by event: every rank refines its own contiguous range of events with no
exchange on the data path.  What crosses ranks is bookkeeping only: the results are gathered on
rank 0 and the step time is the maximum over ranks.  Works with any torch.distributed backend
(nccl on GPUs, gloo in the CPU tests); holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np


def event_range(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced range [begin, end) of rank `rank`: the first n_events % world ranks get one more."""
    if world <= 0 or not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad rank/world/n_events")
    base, extra = divmod(n_events, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def csr_slice(hit_offsets: np.ndarray, begin: int, end: int):
    """Hits of events [begin, end): (first hit, last hit, offsets rebased to 0)."""
    off = np.asarray(hit_offsets, np.int64)
    first, last = int(off[begin]), int(off[end])
    return first, last, (off[begin:end + 1] - first).astype(np.int32)


def max_over_ranks(seconds: float, dist=None, device=None) -> float:
    """Step time of the job = slowest rank.  `dist` = torch.distributed (initialised) or None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(seconds)
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_results(local: np.ndarray, n_events: int, dist=None):
    """Rank 0 receives the per-event result rows of every rank in event order; other ranks get None."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    parts = [None] * world if rank == 0 else None
    dist.gather_object(np.ascontiguousarray(local), parts, dst=0)
    if rank != 0:
        return None
    out = np.concatenate(parts, axis=0)
    if out.shape[0] != n_events:
        raise RuntimeError(f"gathered {out.shape[0]} events, expected {n_events}")
    return out
