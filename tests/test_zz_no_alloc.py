"""ia_topk_static: the top-K for callers that are not allowed to allocate device memory.

Who that is (include/ia.h has the long form): a process whose framework pool owns the whole GPU, a latency-bound event
loop that cannot afford cudaMalloc's device-wide synchronisation, and code running inside a stream capture.  The ordinary
ia_topk grows a buffer of its context on demand; this entry point keeps the same per-block candidate lists in a fixed
256 KB array of the library's device image, takes no context, and leaves inputs and outputs to the caller.

The file sorts after every other test file on purpose: `pytest -x` stops at the first failure, so a problem here cannot
hide the rest of the suite.  The GPU test makes no assumption about what ran before it - it passes alone in a fresh
process (where its first call is the one that looks the array up on the device) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2401_04576_b200 import binding as b


def _accumulator(n, seed, mode):
    rng = np.random.default_rng(seed)
    if mode == "bell":              # the entry bar of the K best rises slowly: many lists carry real candidates
        v = np.clip(rng.normal(12.0, 6.0, n), 0, 60).astype(np.int64)
    elif mode == "plateau":         # ties on the vote count: the order among them is by index
        v = np.where(rng.random(n) < 0.4, 40, rng.integers(0, 40, n))
    else:                           # nearly empty, a few isolated peaks
        v = np.zeros(n, np.int64)
        pos = rng.integers(0, n, max(1, n // 997))
        v[pos] = rng.integers(1, 200, len(pos))
    return v.astype(np.uint16)


@pytest.mark.gpu
def test_static_topk_equals_ia_topk_on_consecutive_calls():
    """Back-to-back calls that share the fixed array: a large accumulator (many blocks, every list in use), then
    smaller ones with other contents (fewer lists: whatever the earlier call left in the array must not show), then
    the first again.  Integer work, so the bar is the one of the other top-K tests: identical indices and counts."""
    import torch
    torch.cuda.set_device(0)
    cases = [((1 << 23) + 77, 10, "bell"), (100003, 32, "plateau"), (4096, 16, "sparse"), (31, 5, "plateau"),
             ((1 << 23) + 77, 10, "bell")]
    host = [_accumulator(n, 1000 + i if i < 4 else 1000, mode) for i, (n, k, mode) in enumerate(cases)]
    dev = [torch.from_numpy(v.view(np.int16)).cuda().view(torch.uint16) for v in host]
    # the caller's outputs exist before the first call; a canary behind the k entries shows nothing is written past them
    idx = [torch.full((k + 4,), -7, dtype=torch.int64, device="cuda") for _, k, _ in cases]
    cnt = [torch.full((k + 4,), 9, dtype=torch.int16, device="cuda").view(torch.uint16) for _, k, _ in cases]
    torch.cuda.synchronize()
    # first call on this device in a fresh process: includes the look-up of the array's device address
    b.ia_topk_static(dev[0], cases[0][1], idx[0], cnt[0])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    for i in range(1, len(cases)):
        b.ia_topk_static(dev[i], cases[i][1], idx[i], cnt[i])
    torch.cuda.synchronize()
    # device-wide free memory did not move across four calls: nothing was allocated (or freed) anywhere on the GPU
    assert torch.cuda.mem_get_info(0)[0] == free_before
    ctx = b.Context(0)
    try:
        for i, (n, k, mode) in enumerate(cases):
            eidx, ecnt = ctx.ia_topk(dev[i], k)
            ctx.synchronize()
            assert (idx[i][:k] == eidx).all() and (cnt[i][:k].view(torch.int16) == ecnt.view(torch.int16)).all(), (i, n, k, mode)
            assert (idx[i][k:] == -7).all() and (cnt[i][k:].view(torch.int16) == 9).all(), "wrote past the k entries"
            # and the definition itself: votes descending, index ascending
            order = np.lexsort((np.arange(n), -host[i].astype(np.int64)))[:k]
            assert (idx[i][:k].cpu().numpy() == order).all() and (cnt[i][:k].cpu().numpy().view(np.uint16) == host[i][order]).all()
        # an accumulator that does not start on a 16-byte boundary, and an explicit stream
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        b.ia_topk_static(dev[1][3:], 8, idx[1], cnt[1], n_cells=cases[1][0] - 3, stream=s)
        s.synchronize()
        eidx, ecnt = ctx.ia_topk(dev[1][3:], 8, n_cells=cases[1][0] - 3)
        ctx.synchronize()
        assert (idx[1][:8] == eidx).all() and (cnt[1][:8].view(torch.int16) == ecnt.view(torch.int16)).all()
    finally:
        ctx.close()


def test_static_topk_names_the_limit_it_refuses():
    """Sizes beyond the stated maxima are refused before any CUDA call is made (so this runs without a GPU), with a
    message that names the limit; the pointers are never dereferenced on the host."""
    lib = b.load_library()
    fake = C.c_void_p(0x1000)

    def call(n_cells, k, votes=fake, idx=fake, cnt=fake):
        rc = lib.ia_topk_static(0, None, votes, n_cells, k, idx, cnt)
        return rc, lib.ia_topk_static_error().decode()

    rc, msg = call(b.TOPK_STATIC_MAX_CELLS + 1, 4)
    assert rc == -4 and "IA_TOPK_STATIC_MAX_CELLS" in msg and str(b.TOPK_STATIC_MAX_CELLS + 1) in msg
    rc, msg = call(1000, 33)
    assert rc == -4 and "IA_MAX_K" in msg
    rc, msg = call(0, 1)
    assert rc == -1 and "n_cells" in msg
    rc, msg = call(5, 6)
    assert rc == -1 and "k <= n_cells" in msg
    rc, msg = call(1000, 4, votes=None)
    assert rc == -1 and "NULL" in msg
