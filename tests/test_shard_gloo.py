"""The N>1 host logic on CPU: world_size-2 gloo processes shard events, gather results, reduce the time."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2401_04576_b200 import shard


def test_event_range_partitions_exactly():
    for n in (0, 1, 5, 1024, 1025):
        for world in (1, 2, 3, 8):
            r = [shard.event_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1


def test_csr_slice():
    off = np.array([0, 3, 3, 10, 12], np.int32)
    first, last, sub = shard.csr_slice(off, 1, 3)
    assert (first, last) == (3, 10) and sub.tolist() == [0, 0, 7]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_events, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        b, e = shard.event_range(n_events, rank, world)
        # stand-in for the per-event result rows (params_out): event id in column 0
        local = np.stack([np.arange(b, e, dtype=np.float64), np.full(e - b, float(rank))], axis=1)
        t = shard.max_over_ranks(0.5 + rank, dist)
        out = shard.gather_results(local, n_events, dist)
        if rank == 0:
            q.put((t, out))
        else:
            assert out is None
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world, n_events = 2, 7
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_events, q)) for r in range(world)]
    for p in procs:
        p.start()
    t, out = q.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert t == 1.5                                      # max over ranks
    assert out.shape == (n_events, 2) and (out[:, 0] == np.arange(n_events)).all()
    assert out[:4, 1].tolist() == [0.0] * 4 and out[4:, 1].tolist() == [1.0] * 3


def _keys_worker(rank, world, port, q):
    import torch
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # stand-in for a rank's ia_topk_keys list: 32 int64 "keys" that name the rank
        local = torch.arange(32, dtype=torch.int64) + 1000 * (rank + 1)
        out = shard.gather_key_lists(local, dist)
        if rank == 0:
            q.put(out.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_key_lists_are_gathered_in_rank_order_gloo():
    """the one exchange of the split dense vote: every rank ends up with all lists, rank after rank"""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_keys_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = q.get(timeout=120)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert out.shape == (64,)
    assert (out[:32] == np.arange(32) + 1000).all() and (out[32:] == np.arange(32) + 2000).all()


def test_slab_ranges_tile_the_axis():
    for nx in (1, 3, 8, 64):
        for world in (1, 2, 3, 8):
            r = [shard.slab_range(nx, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nx and all(r[i][1] == r[i + 1][0] for i in range(world - 1))
