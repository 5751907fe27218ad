"""Host-side sharding across ranks.

Independent events: every rank refines its own contiguous range of events with no exchange on the data path; the results
are gathered on rank 0 and the step time is the maximum over ranks.
One event on several GPUs: the dense vote is split along its slowest axis (xc); every rank votes its
slab (ia_vote_slab), reduces it to its K best keys (ia_topk_keys), the key lists - 256 bytes per rank - are all-gathered
(the one exchange of the path) and merged by every rank (ia_merge_keys).  Works with any torch.distributed backend (nccl
on GPUs, gloo in the CPU tests); holds none of the method's arithmetic: votes, keys and the merge are the library's.
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


def slab_range(nx: int, rank: int, world: int) -> tuple[int, int]:
    """xc cells [begin, end) of rank `rank` in a dense vote split over `world` ranks (balanced, contiguous; a rank may get
    none when world > nx)."""
    return event_range(nx, rank, world)


def gather_key_lists(keys_local, dist=None):
    """All-gather of the per-rank key lists (ia_topk_keys: IA_KEY_LIST uint64 carried as int64) -> one tensor
    [world * IA_KEY_LIST] in rank order on every rank.  A rank with an empty slab contributes zeros (empty keys)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return keys_local
    import torch
    world = dist.get_world_size()
    out = torch.empty(world * keys_local.numel(), dtype=keys_local.dtype, device=keys_local.device)
    dist.all_gather_into_tensor(out, keys_local.contiguous())
    return out


def split_vote_topk(ctx, hits_dev, n_hits, box_lo, box_hi, grid_dims, k, rank=0, world=1, dist=None, votes_out=None):
    """The K best cells of ONE event's dense vote computed by `world` GPUs: slab vote, local key list, all-gather, merge.
    Returns (idx[k], votes[k]) - identical on every rank and identical to ia_vote + ia_topk on one GPU - and the rank's
    slab accumulator.  Every step is a call of the C ABI on ctx's stream, and the all-gather is issued with that stream
    current, so the three are ordered on one stream for any stream the context was built with."""
    import torch
    dims = [int(d) for d in grid_dims]
    b, e = slab_range(dims[0], rank, world)
    col = 1
    for d in dims[1:]:
        col *= d
    if e > b:
        votes = ctx.ia_vote_slab(hits_dev, n_hits, box_lo, box_hi, dims, b, e, votes_out=votes_out)
        keys = ctx.ia_topk_keys(votes, min(k, (e - b) * col), index_base=b * col, n_cells=(e - b) * col)
    else:
        votes = None
        keys = torch.zeros(32, dtype=torch.int64, device=f"cuda:{ctx.device}")
    # the collective is ordered against torch's CURRENT stream only; the C-ABI calls before and after it run on ctx's
    # stream.  Making ctx's stream current for the gather puts all three on one stream, whatever stream the context has.
    if keys.is_cuda and getattr(ctx, "stream", None) is not None:
        with torch.cuda.stream(ctx.stream):
            all_keys = gather_key_lists(keys, dist)
    else:
        all_keys = gather_key_lists(keys, dist)
    idx, v = ctx.ia_merge_keys(all_keys, all_keys.numel() // 32, k)
    return idx, v, votes
