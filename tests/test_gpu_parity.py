"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element.

Bars (BASELINE.json north_star): top-K boxes and recovered parameters identical at every level;
vote accumulator equal in >= 99.99 % of cells with every mismatch traced to a residual endpoint
within 1e-12 relative of zero; integer/index work bit-exact.
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import binding as b
from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

from gpu_common import HI, LO, Rig, compare_votes

pytestmark = pytest.mark.gpu

ADD, SUB, MUL, SQR, DIV, SQRT, SIN, COS, ATAN2, RECIP, SCALE = range(11)


@pytest.fixture(scope="module")
def rig0():
    r = Rig(g.chamber_c0())
    yield r
    r.close()


@pytest.fixture(scope="module")
def rig1():
    r = Rig(g.chamber_c1())
    yield r
    r.close()


def _rand_iv(rng, n, positive=False, prec=64):
    m = rng.choice([1e-3, 1.0, 37.0, 450.0, 1e5], size=n)
    a, c = rng.uniform(-m, m), rng.uniform(-m, m)
    lo, hi = np.minimum(a, c), np.maximum(a, c)
    thin = rng.random(n) < 0.15
    hi = np.where(thin, lo, hi)
    if positive:
        lo, hi = np.abs(lo) + 1e-3, np.abs(hi) + 1e-3
        lo, hi = np.minimum(lo, hi), np.maximum(lo, hi)
    if prec == 32:
        lo, hi = lo.astype(np.float32).astype(np.float64), hi.astype(np.float32).astype(np.float64)
        lo, hi = np.minimum(lo, hi), np.maximum(lo, hi)
    return np.stack([lo, hi], 1)


@pytest.mark.parametrize("prec", [64, 32])
def test_arithmetic_primitives_bit_exact(rig0, prec):
    """Both sides return the tightest enclosure, so + - * sqr / sqrt recip scale agree bit for bit."""
    rng = np.random.default_rng(prec)
    n = 3000
    a, bb, bp = _rand_iv(rng, n, prec=prec), _rand_iv(rng, n, prec=prec), _rand_iv(rng, n, True, prec)
    # sign cases with zeros and signed zeros
    pts = [-3.5, -1.25, -0.0, 0.0, 0.75, 2.5]
    ivs = np.array([(x, y) for x in pts for y in pts if x <= y])
    a[: len(ivs) ** 2] = np.repeat(ivs, len(ivs), 0)
    bb[: len(ivs) ** 2] = np.tile(ivs, (len(ivs), 1))
    ctx = rig0.ctx
    for op, x, y in ((ADD, a, bb), (SUB, a, bb), (MUL, a, bb), (SQR, a, None), (DIV, a, bp), (SQRT, bp, None),
                     (RECIP, bp, None), (SCALE, a, bb)):
        got = ctx.ia_prim(op, prec, rig0.dev(x), None if y is None else rig0.dev(y)).cpu().numpy()
        for i in range(n):
            yy = (0.0, 0.0) if y is None else tuple(y[i])
            if op == SCALE:
                yy = (y[i, 0], y[i, 0])
            exp = o.prim(op, tuple(x[i]), yy, prec)
            assert (got[i, 0] == exp[0] and got[i, 1] == exp[1]) or (np.isnan(exp[0]) and np.isnan(got[i, 0])), (op, x[i], yy, got[i], exp)


@pytest.mark.parametrize("prec", [64, 32])
def test_elementary_enclosures(rig0, prec):
    """sin/cos/atan2: the GPU enclosure overlaps the oracle's everywhere, both within their pads:
    |gpu - oracle| <= (pad_gpu + pad_oracle + 2) ulps at each endpoint, same special cases."""
    rng = np.random.default_rng(3)
    n = 4000
    eps = 2.0 ** -52 if prec == 64 else 2.0 ** -23
    w = rng.choice([0.0, 1e-9, 1e-3, 0.1, 1.0, 3.0], size=n)
    c = rng.uniform(-4.5, 4.5, n)
    e = np.stack([c - w, c + w], 1)
    if prec == 32:
        e = e.astype(np.float32).astype(np.float64)
    y, x = _rand_iv(rng, n, prec=prec), _rand_iv(rng, n, prec=prec)
    ctx = rig0.ctx
    tol_ulps = 8 + o.pad_ulps() + 2
    for op, A, B, mag in ((SIN, e, None, 1.0), (COS, e, None, 1.0), (ATAN2, y, x, 4.0)):
        got = ctx.ia_prim(op, prec, rig0.dev(A), None if B is None else rig0.dev(B)).cpu().numpy()
        for i in range(n):
            exp = o.prim(op, tuple(A[i]), (0.0, 0.0) if B is None else tuple(B[i]), prec)
            assert abs(got[i, 0] - exp[0]) <= tol_ulps * eps * mag and abs(got[i, 1] - exp[1]) <= tol_ulps * eps * mag, \
                (op, A[i], got[i], exp)
            assert got[i, 0] <= exp[1] and exp[0] <= got[i, 1]
            if exp in ((-1.0, 1.0),) or abs(exp[1]) == 1.0 or abs(exp[0]) == 1.0:
                pass
        # exact special values
    sp = np.array([[-5.0, 0.0], [0.0, 4.5], [1.0, 2.0], [-2.0, -1.0], [-0.5, 0.25], [3.0, 3.5]])
    s = ctx.ia_prim(SIN, prec, rig0.dev(sp)).cpu().numpy()
    cc = ctx.ia_prim(COS, prec, rig0.dev(sp)).cpu().numpy()
    assert tuple(s[0]) == (-1.0, 1.0) and tuple(cc[1]) == (-1.0, 1.0)
    assert s[2, 1] == 1.0 and s[3, 0] == -1.0 and cc[4, 1] == 1.0 and cc[5, 0] == -1.0
    cut = ctx.ia_prim(ATAN2, prec, rig0.dev(np.array([[-1.0, 1.0]])), rig0.dev(np.array([[-2.0, -1.0]]))).cpu().numpy()
    assert tuple(cut[0]) == o.prim(ATAN2, (-1.0, 1.0), (-2.0, -1.0), prec)


def _random_boxes(rng, n, min_log2=2, max_log2=12):
    c = rng.uniform(LO * 0.9 + HI * 0.1, LO * 0.1 + HI * 0.9, size=(n, 5))
    w = (HI - LO) * 2.0 ** -rng.integers(min_log2, max_log2, size=(n, 1))
    blo, bhi = c - w / 2, c + w / 2
    blo[:, 2] = np.maximum(blo[:, 2], 20.0)
    blo[:, 4], bhi[:, 4] = np.maximum(blo[:, 4], -0.6), np.minimum(bhi[:, 4], 0.6)
    return blo, bhi


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("ref", [(0.0, 0.0, 0.0), (1.5, -2.0, 3.0)])
def test_residual_enclosures_match(precision, ref):
    """f enclosures of random (box, hit, sign): endpoints agree to a few ulps of the residual's scale."""
    rng = np.random.default_rng(11)
    rig = Rig(g.chamber_c1(), precision=precision, x_ref=ref[0], y_ref=ref[1], z_ref=ref[2])
    try:
        ev = g.make_event(rig.ch, 5, n_noise=12)
        hd, oh = rig.hits(ev.wire, ev.drift)
        blo, bhi = _random_boxes(rng, 600)
        # boxes around the truth as well, where the enclosures are tight and straddle zero
        par = np.array(ev.track.params)
        for i in range(0, 200):
            half = (HI - LO) * 2.0 ** -rng.integers(6, 14) / 2
            cc = par + rng.uniform(-1, 1, 5) * half
            blo[i], bhi[i] = cc - half, cc + half
        rg = rig.gpu_residual(hd, len(oh), blo, bhi)
        ro = o.residual(rig.owires, oh, rig.oparams, blo, bhi)
        assert (rg[..., 3] == ro[..., 3]).all()
        live = ro[..., 3] == 0
        tol = (1e-13 if precision == 64 else 2e-4) * ro[..., 2]
        assert (np.abs(rg[..., 0] - ro[..., 0])[live] <= tol[live]).all()
        assert (np.abs(rg[..., 1] - ro[..., 1])[live] <= tol[live]).all()
        assert np.allclose(rg[..., 2][live], ro[..., 2][live], rtol=1e-6 if precision == 64 else 1e-3)
        vg = (rg[..., 3] == 1) | ((rg[..., 0] <= 0) & (rg[..., 1] >= 0))
        vo = (ro[..., 3] == 1) | ((ro[..., 0] <= 0) & (ro[..., 1] >= 0))
        assert (vg == vo).mean() > 0.9999 and vg.any() and not vg.all()
    finally:
        rig.close()


def test_c0_dense_vote_full_parity(rig0):
    """configs[0]: 16^5 cells x 8 hits, every cell compared."""
    cfg = g.config(0)
    ev = cfg.events[0]
    hd, oh = rig0.hits(ev.wire, ev.drift)
    vg = rig0.ctx.ia_vote(hd, ev.n_hits, LO, HI, cfg.grid)
    rig0.ctx.synchronize()
    vg = vg.cpu().numpy()
    vo = o.vote(rig0.owires, oh, rig0.oparams, LO, HI, cfg.grid)
    n_bad = compare_votes(rig0, hd, oh, vg, vo, lambda idx: o.cell_boxes(LO, HI, cfg.grid, idx))
    assert vg.max() == 8 and n_bad <= len(vg) // 10000
    truth = g.truth_cell(ev.track.params, LO, HI, cfg.grid)
    assert vg[truth] >= (~ev.clipped).sum() - 1       # smeared hits: 3-sigma tolerance, allow one miss


@pytest.mark.parametrize("dims", [(3, 5, 7, 2, 9), (1, 1, 1, 1, 1), (2, 2, 33, 17, 6), (6, 4, 3, 130, 5)])
def test_ragged_grids(rig0, dims):
    """Grid shapes that do not divide the block tiling, with a lambda cell straddling 0 (odd n)."""
    ev = g.make_event(rig0.ch, 7, n_noise=3)
    hd, oh = rig0.hits(ev.wire, ev.drift)
    vg = rig0.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
    rig0.ctx.synchronize()
    vo = o.vote(rig0.owires, oh, rig0.oparams, LO, HI, dims)
    # the 99.99 % bar needs >= 10^4 cells to allow a single (traced) knife-edge cell; the two small grids get one
    compare_votes(rig0, hd, oh, vg.cpu().numpy(), vo, lambda idx: o.cell_boxes(LO, HI, dims, idx),
                  min_equal=0.9999 if np.prod(dims) >= 10000 else 1.0 - 1.5 / np.prod(dims))


def test_small_window_grid_around_truth(rig1):
    """A fine grid around the truth (cells of range/2048): votes vary cell to cell here."""
    ev = g.make_event(rig1.ch, 21, n_noise=5)
    hd, oh = rig1.hits(ev.wire, ev.drift)
    par = np.array(ev.track.params)
    half = (HI - LO) / 256
    lo, hi = par - half, par + half
    dims = (8, 8, 8, 8, 8)
    vg = rig1.ctx.ia_vote(hd, ev.n_hits, lo, hi, dims)
    rig1.ctx.synchronize()
    vg = vg.cpu().numpy()
    vo = o.vote(rig1.owires, oh, rig1.oparams, lo, hi, dims)
    compare_votes(rig1, hd, oh, vg, vo, lambda idx: o.cell_boxes(lo, hi, dims, idx))
    assert len(np.unique(vg)) > 4


def test_vote_boxes_and_empty_inputs(rig1):
    rng = np.random.default_rng(2)
    ev = g.make_event(rig1.ch, 9, n_noise=20)
    hd, oh = rig1.hits(ev.wire, ev.drift)
    blo, bhi = _random_boxes(rng, 1000, 2, 10)
    vg = rig1.ctx.ia_vote_boxes(hd, ev.n_hits, rig1.dev(blo), rig1.dev(bhi))
    rig1.ctx.synchronize()
    vo = o.vote_boxes(rig1.owires, oh, rig1.oparams, blo, bhi)
    # 1,000 boxes: one traced knife-edge box allowed (the 99.99 % bar needs 10^4)
    compare_votes(rig1, hd, oh, vg.cpu().numpy(), vo, lambda idx: (blo[idx], bhi[idx]), min_equal=0.999, kind="boxes")
    # no hits: all zero
    v0 = rig1.ctx.ia_vote(None, 0, LO, HI, (4, 4, 4, 4, 4))
    rig1.ctx.synchronize()
    assert int(v0.cpu().numpy().astype(np.int64).sum()) == 0


# (1 << 23) + 77 cells: beyond the size from which the streaming form (8 loads in flight per lane) is taken
@pytest.mark.parametrize("n,k", [(1, 1), (31, 5), (32, 32), (257, 10), (4096, 16), (100003, 8), (1 << 21, 10),
                                 ((1 << 23) + 77, 10), ((1 << 23) + 77, 32)])
def test_topk_bit_exact(rig0, n, k):
    import torch
    rng = np.random.default_rng(n)
    for mode in ("random", "plateau", "zeros", "late_peak", "ramp", "bell", "sparse"):
        if mode == "random":
            v = rng.integers(0, 41, n)
        elif mode == "plateau":
            v = np.where(rng.random(n) < 0.4, 40, rng.integers(0, 40, n))
        elif mode == "zeros":
            v = np.zeros(n, np.int64)
        elif mode == "ramp":            # rising: every chunk beats the entry bar (single-key insertions all the way)
            v = (np.arange(n, dtype=np.int64) * 60000) // max(n, 1) + rng.integers(0, 3, n)
        elif mode == "bell":            # the entry bar rises slowly (many rare records)
            v = np.clip(rng.normal(12.0, 6.0, n), 0, 60).astype(np.int64)
        elif mode == "sparse":          # one or two lanes of a chunk above the bar
            v = np.zeros(n, np.int64)
            pos = rng.integers(0, n, max(1, n // 997))
            v[pos] = rng.integers(1, 200, len(pos))
        else:
            v = rng.integers(0, 5, n)
            v[-min(n, 3):] = 60
        v = v.astype(np.uint16)
        vd = torch.from_numpy(v.view(np.int16)).cuda().view(torch.uint16)
        idx, vv = rig0.ctx.ia_topk(vd, k)
        rig0.ctx.synchronize()
        eidx, ev = o.topk(v, k)
        assert (idx.cpu().numpy() == eidx).all() and (vv.cpu().numpy() == ev).all(), (n, k, mode)
    # unaligned view: the 16-byte path must not be taken blindly
    if n > 64:
        v = rng.integers(0, 41, n).astype(np.uint16)
        vd = torch.from_numpy(v.view(np.int16)).cuda().view(torch.uint16)
        idx, vv = rig0.ctx.ia_topk(vd[3:], k, n_cells=n - 3)
        rig0.ctx.synchronize()
        eidx, ev = o.topk(v[3:], k)
        assert (idx.cpu().numpy() == eidx).all() and (vv.cpu().numpy() == ev).all()


def _assert_boxes_equal(gb, ob):
    assert (gb["lo"] == ob["lo"]).all() and (gb["hi"] == ob["hi"]).all(), "boxes differ"
    assert (gb["votes"] == ob["votes"]).all(), "votes differ"


def test_c2_refine_identical_at_every_level(rig1):
    """configs[2]: 8^5 start, K=16, 10 passes: the kept boxes and the parameters are identical."""
    cfg = g.config(2)
    ev = cfg.events[0]
    hd, oh = rig1.hits(ev.wire, ev.drift)
    boxes, par = rig1.ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, cfg.levels, cfg.k)
    rig1.ctx.synchronize()
    gb = b.boxes_to_numpy(boxes, (cfg.levels, cfg.k))
    ob, opar = o.refine(rig1.owires, oh, rig1.oparams, LO, HI, cfg.grid, cfg.levels, cfg.k)
    _assert_boxes_equal(gb, ob)
    assert (par.cpu().numpy() == opar).all()
    assert np.all(opar[5:10] * 2 < (HI - LO) * 1e-3)            # final box width < 1e-3 of the range


@pytest.mark.parametrize("precision", [64, 32])
def test_c3_refine_batch_identical(precision):
    """configs[3] shape (8^5 start, K=8, 8 passes) on a handful of events, FP64 and FP32 intervals."""
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        cfg = g.config(3, n_events=5)
        wire = np.concatenate([e.wire for e in cfg.events])
        drift = np.concatenate([e.drift for e in cfg.events])
        off = np.cumsum([0] + [e.n_hits for e in cfg.events]).astype(np.int32)
        hd, oh = rig.hits(wire, drift)
        boxes, par = rig.ctx.ia_refine_batch(hd, rig.dev(off), len(cfg.events), 30, LO, HI, cfg.grid, cfg.levels, cfg.k)
        rig.ctx.synchronize()
        gb = b.boxes_to_numpy(boxes, (len(cfg.events), cfg.levels, cfg.k))
        ob, opar = o.refine_batch(rig.owires, oh, off, rig.oparams, LO, HI, cfg.grid, cfg.levels, cfg.k)
        _assert_boxes_equal(gb, ob)
        assert (par.cpu().numpy().reshape(-1, 20) == opar).all()
        # host-buffer entry point gives the same answer
        hb, hp = rig.ctx.ia_refine_batch_host(b.hits_of(wire, drift), off, LO, HI, cfg.grid, cfg.levels, cfg.k)
        _assert_boxes_equal(hb, ob)
        assert (hp == opar).all()
    finally:
        rig.close()


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("grid,levels,k", [((8,) * 5, 6, 8), ((4, 4, 4, 4, 5), 5, 3), ((6, 5, 4, 3, 2), 4, 32),
                                           ((3, 3, 3, 3, 3), 7, 1)])
def test_children_fast_and_general_kernels_agree(precision, grid, levels, k):
    """The sign-specialised children kernel against the general one (IA_FLAG_GENERAL) and against the oracle:
    K = 3 and 1 leave warps partly filled, an odd lambda grid makes parents whose children straddle 0,
    K = 32 is the largest list."""
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        evs = [g.make_event(rig.ch, 2000 + e, n_noise=6) for e in range(3)]
        wire = np.concatenate([e.wire for e in evs])
        drift = np.concatenate([e.drift for e in evs])
        off = np.cumsum([0] + [e.n_hits for e in evs]).astype(np.int32)
        hd, oh = rig.hits(wire, drift)
        mh = max(e.n_hits for e in evs)
        out = []
        for flags in (0, b.FLAG_GENERAL):
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=flags)
            boxes, par = rig.ctx.ia_refine_batch(hd, rig.dev(off), len(evs), mh, LO, HI, grid, levels, k)
            rig.ctx.synchronize()
            out.append((b.boxes_to_numpy(boxes, (len(evs), levels, k)), par.cpu().numpy().reshape(-1, 20)))
        ob, opar = o.refine_batch(rig.owires, oh, off, rig.oparams, LO, HI, grid, levels, k)
        _assert_boxes_equal(out[0][0], out[1][0])
        _assert_boxes_equal(out[0][0], ob)
        assert (out[0][1] == opar).all() and (out[1][1] == opar).all()
    finally:
        rig.close()


def test_c1_dense_vote_sampled_and_top10(rig1):
    """configs[1]: 32^5 x 40 hits at full size; 30000 sampled cells + the GPU's top-10 cells against
    the oracle, and the top-10 selection itself bit-exact on the GPU's accumulator."""
    cfg = g.config(1)
    ev = cfg.events[0]
    hd, oh = rig1.hits(ev.wire, ev.drift)
    votes = rig1.ctx.ia_vote(hd, ev.n_hits, LO, HI, cfg.grid)
    idx, vv = rig1.ctx.ia_topk(votes, cfg.k)
    rig1.ctx.synchronize()
    vg = votes.cpu().numpy()
    eidx, evv = o.topk(vg, cfg.k)
    assert (idx.cpu().numpy() == eidx).all() and (vv.cpu().numpy() == evv).all()
    rng = np.random.default_rng(1)
    sample = np.unique(np.concatenate([rng.integers(0, cfg.n_cells, 30000), eidx,
                                       [g.truth_cell(ev.track.params, LO, HI, cfg.grid)],
                                       np.nonzero(vg == vg.max())[0][:2000]]))
    vo = o.vote(rig1.owires, oh, rig1.oparams, LO, HI, cfg.grid, cell_idx=sample)
    compare_votes(rig1, hd, oh, vg[sample], vo, lambda i: o.cell_boxes(LO, HI, cfg.grid, sample[i]))
    assert vg.max() <= ev.n_hits


def test_errors_and_device_status(rig0):
    ctx = rig0.ctx
    ev = g.make_event(rig0.ch, 1)
    hd, _ = rig0.hits(ev.wire, ev.drift)
    lo = LO.copy()
    lo[2] = 0.0
    with pytest.raises(b.IaError) as ei:
        ctx.ia_vote(hd, ev.n_hits, lo, HI, (2,) * 5)
    assert ei.value.code == -3
    hi = HI.copy()
    hi[4] = 6.0
    with pytest.raises(b.IaError) as ei:
        ctx.ia_vote(hd, ev.n_hits, LO, hi, (2,) * 5)
    assert ei.value.code == -3
    with pytest.raises(b.IaError) as ei:
        ctx.ia_vote(hd, ev.n_hits, HI, LO, (2,) * 5)
    assert ei.value.code == -1
    with pytest.raises(b.IaError) as ei:
        ctx.ia_refine(hd, ev.n_hits, LO, HI, (2,) * 5, 2, b.IA_MAX_K + 1)
    assert ei.value.code in (-1, -4)
    with pytest.raises(b.IaError) as ei:
        ctx.ia_vote_host(b.hits_of([99999], [0.3]), LO, HI, (2,) * 5)
    assert ei.value.code == -2
    # a bad wire on the device path: the hit is dropped and the sticky status reports it once
    bad, _ = rig0.hits(np.append(ev.wire, 99999).astype(np.int32), np.append(ev.drift, 0.2))
    v = ctx.ia_vote(bad, ev.n_hits + 1, LO, HI, (4,) * 5)
    with pytest.raises(b.IaError) as ei:
        ctx.ia_device_status()
    assert ei.value.code == -2
    ctx.ia_device_status()
    good = ctx.ia_vote(hd, ev.n_hits, LO, HI, (4,) * 5)
    ctx.synchronize()
    assert (v.cpu().numpy() == good.cpu().numpy()).all()
    # a context without geometry refuses to vote
    c2 = b.Context(0)
    with pytest.raises(b.IaError) as ei:
        c2.ia_vote(hd, ev.n_hits, LO, HI, (2,) * 5)
    assert ei.value.code == -2
    c2.close()


def test_host_entry_point_matches_device_path(rig0):
    ev = g.make_event(rig0.ch, 3, n_noise=2)
    hd, _ = rig0.hits(ev.wire, ev.drift)
    dims = (6, 6, 6, 6, 6)
    vd = rig0.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
    rig0.ctx.synchronize()
    vh = rig0.ctx.ia_vote_host(b.hits_of(ev.wire, ev.drift), LO, HI, dims)
    assert (vd.cpu().numpy() == vh).all()
    assert rig0.ctx.ia_launch_count() > 0
    # accumulators of 32 MB and more leave in slabs of xc cells, copied while the next slab is voted (2 and 3 uneven slabs)
    for dims in ((37, 32, 32, 32, 32), (7, 64, 64, 64, 32)):
        vd = rig0.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
        rig0.ctx.synchronize()
        vh = rig0.ctx.ia_vote_host(b.hits_of(ev.wire, ev.drift), LO, HI, dims)
        assert (vd.cpu().numpy() == vh).all(), dims


@pytest.mark.parametrize("nx,slab_min,n_slabs", [(5, 2000, 2), (7, 2200, 3), (7, 1, 7), (13, 700, 8), (11, 1, 8), (3, 1 << 40, 1)])
def test_host_slab_pipeline_every_cell_on_ragged_grids(rig0, nx, slab_min, n_slabs):
    """The slab pipeline of ia_vote_host (vote of slab i+1 beside the copy of slab i on a second stream) with the slab
    size lowered so that small grids take it: 2, 3, 7 and 8 slabs of unequal width on an odd number of xc cells, every
    cell compared with ia_vote; the buffer between canaries, a second call into the same buffer (the copies of the
    first must be over), and the single-launch path of the same call."""
    ev = g.make_event(rig0.ch, 5, n_noise=3)
    hd, _ = rig0.hits(ev.wire, ev.drift)
    hh = b.hits_of(ev.wire, ev.drift)
    dims = (nx, 3, 6, 7, 9)
    n = int(np.prod(dims))
    assert min(8, nx, n // slab_min) == n_slabs or (n_slabs == 1 and n // slab_min < 2)
    vd = rig0.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
    rig0.ctx.synchronize()
    vd = vd.cpu().numpy()
    assert vd.max() > 0
    launches0 = rig0.ctx.ia_launch_count()
    try:
        rig0.ctx.ia_set_host_slab_min(slab_min)
        buf = np.full(n + 64, 0xA5A5, np.uint16)
        for _ in range(2):
            buf[32:32 + n] = 0xFFFF
            rig0.ctx.ia_vote_host(hh, LO, HI, dims, votes_out=buf[32:32 + n])
            assert (buf[32:32 + n] == vd).all(), (dims, slab_min)
            assert (buf[:32] == 0xA5A5).all() and (buf[32 + n:] == 0xA5A5).all()
        # one staging launch + one vote launch per slab and call (small grids may add a partial-sum launch per slab)
        assert rig0.ctx.ia_launch_count() - launches0 >= 2 * (1 + n_slabs)
    finally:
        rig0.ctx.ia_set_host_slab_min(16 << 20)
    with pytest.raises(b.IaError):
        rig0.ctx.ia_set_host_slab_min(0)


@pytest.mark.parametrize("precision", [64, 32])
def test_fast_and_general_kernels_agree(precision):
    """The sign-specialised dense kernel against the general one (IA_FLAG_GENERAL) on a full 24^5 grid and
    on ragged shapes: same DAG, same roundings, so only the sin/cos pads may move a knife-edge cell."""
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        ev = g.make_event(rig.ch, 31, n_noise=10)
        hd, oh = rig.hits(ev.wire, ev.drift)
        for dims in ((24,) * 5, (5, 4, 10, 9, 12), (3, 3, 6, 20, 7), (2, 2, 64, 3, 64)):
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=0)
            vf = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=b.FLAG_GENERAL)
            vg = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            rig.ctx.synchronize()
            vf, vg = vf.cpu().numpy(), vg.cpu().numpy()
            bad = np.nonzero(vf != vg)[0]
            assert len(bad) <= len(vf) // 100000, (dims, len(bad), bad[:10], vf[bad[:10]], vg[bad[:10]])
            assert vf.max() > 0
    finally:
        rig.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_one_body_and_three_body_variants_identical(precision):
    """The two compiled forms of the sign-specialised dense kernel (IA_FLAG_ONE_BODY: sign class as a run-time
    value in one body; bit 2: three bodies) do the same arithmetic: votes identical bit for bit, on a
    coarse and on a fine grid, and whichever the library picks by itself equals both."""
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        ev = g.make_event(rig.ch, 33, n_noise=10)
        hd, oh = rig.hits(ev.wire, ev.drift)
        for dims in ((8,) * 5, (20, 20, 12, 9, 12), (3, 3, 6, 20, 7)):
            out = []
            for flags in (b.FLAG_ONE_BODY, b.FLAG_THREE_BODY, 0):
                rig.ctx.ia_set_params(g.TOL, precision=precision, flags=flags)
                out.append(rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims))
            rig.ctx.synchronize()
            a, c, d = (t.cpu().numpy() for t in out)
            assert (a == c).all() and (a == d).all(), dims
            assert a.max() > 0
    finally:
        rig.close()


PROD_P, PROD_U, D_OVER_SQRT, SQR_U, SIN_SMALL, COS_SMALL, CLAMP_UNIT, SIN_MEDIUM, COS_MEDIUM = 11, 12, 13, 14, 15, 16, 17, 18, 19


@pytest.mark.parametrize("prec", [64, 32])
def test_fast_path_primitives(rig0, prec):
    """The primitives of the dense fast path (ia_fast.cuh) against exact arithmetic: every result
    contains the exact range and is at most a few ulps wider than the tightest enclosure."""
    from fractions import Fraction as Fr
    import mpmath as mp
    mp.mp.dps = 60
    rng = np.random.default_rng(100 + prec)
    n = 1500
    eps = 2.0 ** -52 if prec == 64 else 2.0 ** -23
    ctx = rig0.ctx
    x, ap, au = _rand_iv(rng, n, prec=prec), _rand_iv(rng, n, True, prec), _rand_iv(rng, n, prec=prec)
    ap[:50, 0] = 0.0                                   # factors touching zero (the first lambda cell)
    x[:25] = np.stack([np.zeros(25), np.abs(x[:25, 1])], 1)
    x[25:50] = np.stack([-np.abs(x[25:50, 0]), -np.zeros(25)], 1)
    for op, a in ((PROD_P, ap), (PROD_U, au)):
        got = ctx.ia_prim(op, prec, rig0.dev(a), rig0.dev(x)).cpu().numpy()
        for i in range(n):
            prods = [Fr(p) * Fr(q) for p in a[i] for q in x[i]]
            lo, hi = min(prods), max(prods)
            scale = max(abs(lo), abs(hi), Fr(1, 10 ** 300))
            assert Fr(got[i, 0]) <= lo and hi <= Fr(got[i, 1]), (op, a[i], x[i], got[i])
            assert lo - Fr(got[i, 0]) <= 4 * Fr(eps) * scale and Fr(got[i, 1]) - hi <= 4 * Fr(eps) * scale, (op, a[i], x[i], got[i])
    # D / sqrt(u2)
    d = np.sort(rng.uniform(0.0, 1.6, size=(n, 2)), axis=1)
    d[:20, 0] = 0.0
    u2 = np.sort(rng.uniform(0.3, 3.0, size=(n, 2)), axis=1)
    u2[:200, 1] = u2[:200, 0]
    if prec == 32:
        d, u2 = d.astype(np.float32).astype(np.float64), u2.astype(np.float32).astype(np.float64)
    got = ctx.ia_prim(D_OVER_SQRT, prec, rig0.dev(d), rig0.dev(u2)).cpu().numpy()
    for i in range(n):
        lo, hi = mp.mpf(d[i, 0]) / mp.sqrt(mp.mpf(u2[i, 1])), mp.mpf(d[i, 1]) / mp.sqrt(mp.mpf(u2[i, 0]))
        assert mp.mpf(got[i, 0]) <= lo and hi <= mp.mpf(got[i, 1]), (d[i], u2[i], got[i])
        assert lo - mp.mpf(got[i, 0]) <= 8 * eps * hi and mp.mpf(got[i, 1]) - hi <= 8 * eps * hi, (d[i], u2[i], got[i])
    # branch-free square and the clamp: bit-exact
    got = ctx.ia_prim(SQR_U, prec, rig0.dev(au)).cpu().numpy()
    for i in range(n):
        assert tuple(got[i]) == o.prim(SQR, tuple(au[i]), (0.0, 0.0), prec)
    cl = np.concatenate([_rand_iv(rng, 300, prec=prec) * 1e-2, np.array([[-1.0, 1.0], [-1.0 - 4 * eps, 1.0 + 4 * eps], [-0.0, 0.0], [1.0 - eps, 1.0 + eps]])])
    if prec == 32:
        cl = cl.astype(np.float32).astype(np.float64)
    got = ctx.ia_prim(CLAMP_UNIT, prec, rig0.dev(cl)).cpu().numpy()
    assert (got[:, 0] == np.maximum(cl[:, 0], -1.0)).all() and (got[:, 1] == np.minimum(cl[:, 1], 1.0)).all()
    # sin / cos inside [-1/4, 1/4]
    c = rng.uniform(-0.25, 0.25, n)
    w = rng.choice([0.0, 1e-12, 1e-6, 1e-3, 0.05, 0.5], size=n) * rng.random(n)
    e = np.clip(np.stack([c - w, c + w], 1), -0.25, 0.25)
    e[:10] = [[-0.25, 0.25]] * 10
    e[10:20] = np.stack([np.zeros(10), np.abs(e[10:20, 1])], 1)
    e[20:30] = np.stack([-np.abs(e[20:30, 0]), -np.zeros(10)], 1)
    if prec == 32:
        e = e.astype(np.float32).astype(np.float64)
    s = ctx.ia_prim(SIN_SMALL, prec, rig0.dev(e)).cpu().numpy()
    cc = ctx.ia_prim(COS_SMALL, prec, rig0.dev(e)).cpu().numpy()
    for i in range(n):
        lo, hi = mp.mpf(e[i, 0]), mp.mpf(e[i, 1])
        assert mp.mpf(s[i, 0]) <= mp.sin(lo) and mp.sin(hi) <= mp.mpf(s[i, 1]), (e[i], s[i])
        assert mp.sin(lo) - mp.mpf(s[i, 0]) <= 10 * eps * 0.25 and mp.mpf(s[i, 1]) - mp.sin(hi) <= 10 * eps * 0.25, (e[i], s[i])
        cmin = mp.cos(max(abs(lo), abs(hi)))
        cmax = mp.mpf(1) if lo <= 0 <= hi else mp.cos(min(abs(lo), abs(hi)))
        assert mp.mpf(cc[i, 0]) <= cmin and cmax <= mp.mpf(cc[i, 1]) and cc[i, 1] <= 1.0, (e[i], cc[i])
        assert cmin - mp.mpf(cc[i, 0]) <= 10 * eps and mp.mpf(cc[i, 1]) - cmax <= 10 * eps, (e[i], cc[i])
    # the medium tier: sin / cos inside (-1, 1) by the longer polynomials - contains the truth, and is at most 10 ulps of
    # the result (sin) / of 1 (cos) wider: the relative pad 2^-50 (2^-21) = 8 half-ulps plus the polynomial's own error
    if True:
        c = rng.uniform(-1.0, 1.0, n)
        w = rng.choice([0.0, 1e-12, 1e-6, 1e-3, 0.05, 0.5, 2.0], size=n) * rng.random(n)
        lim = float(np.nextafter(1.0, 0.0)) if prec == 64 else float(np.nextafter(np.float32(1.0), np.float32(0.0)))
        e = np.clip(np.stack([c - w, c + w], 1), -lim, lim)
        if prec == 32:
            e = np.clip(e.astype(np.float32).astype(np.float64), -lim, lim)
        e[:10] = [[-lim, lim]] * 10
        e[10:20] = np.stack([np.zeros(10), np.abs(e[10:20, 1])], 1)
        e[20:30] = np.stack([-np.abs(e[20:30, 0]), -np.zeros(10)], 1)
        e[30:40] = [[lim, lim]] * 10
        s = ctx.ia_prim(SIN_MEDIUM, prec, rig0.dev(e)).cpu().numpy()
        cc = ctx.ia_prim(COS_MEDIUM, prec, rig0.dev(e)).cpu().numpy()
        for i in range(n):
            lo, hi = mp.mpf(e[i, 0]), mp.mpf(e[i, 1])
            assert mp.mpf(s[i, 0]) <= mp.sin(lo) and mp.sin(hi) <= mp.mpf(s[i, 1]), (e[i], s[i])
            assert mp.sin(lo) - mp.mpf(s[i, 0]) <= 10 * eps * max(abs(mp.sin(lo)), mp.mpf(2) ** -1000), (e[i], s[i])
            assert mp.mpf(s[i, 1]) - mp.sin(hi) <= 10 * eps * max(abs(mp.sin(hi)), mp.mpf(2) ** -1000), (e[i], s[i])
            cmin = mp.cos(max(abs(lo), abs(hi)))
            cmax = mp.mpf(1) if lo <= 0 <= hi else mp.cos(min(abs(lo), abs(hi)))
            assert mp.mpf(cc[i, 0]) <= cmin and cmax <= mp.mpf(cc[i, 1]) and cc[i, 1] <= 1.0, (e[i], cc[i])
            assert cmin - mp.mpf(cc[i, 0]) <= 10 * eps and mp.mpf(cc[i, 1]) - cmax <= 10 * eps, (e[i], cc[i])
            # the polynomial alone stays well inside the pad: the padded endpoint is at least 2 half-ulps beyond the truth
            assert mp.sin(hi) - mp.mpf(s[i, 1]) <= 0 and cmin - mp.mpf(cc[i, 0]) >= 2 * (eps / 2) * cmin, (e[i], cc[i])


def test_refine_graph_replay_gives_the_same_boxes(rig1):
    """ia_refine repeated with identical arguments is replayed as a CUDA graph from the third call on: results
    identical to the direct path (IA_FLAG_NO_GRAPH), also after the hits in the same buffer change, after another call
    in between, and with new output buffers."""
    cfg = g.config(2)
    ev = cfg.events[0]
    hd, oh = rig1.hits(ev.wire, ev.drift)
    ctx = rig1.ctx
    ctx.ia_set_params(g.TOL, flags=b.FLAG_NO_GRAPH)
    b0, p0 = ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k)
    ctx.synchronize()
    ref = (b.boxes_to_numpy(b0, (5, cfg.k)).copy(), p0.cpu().numpy().copy())
    ctx.ia_set_params(g.TOL, flags=0)
    boxes, par = ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k)
    n_direct = None
    for i in range(5):
        l0 = ctx.ia_launch_count()
        ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k, boxes=boxes, params=par)
        ctx.synchronize()
        n = ctx.ia_launch_count() - l0
        n_direct = n if n_direct is None else n_direct
        assert n == n_direct                                   # the launch count is the same on every path
        gb = b.boxes_to_numpy(boxes, (5, cfg.k))
        assert (gb["lo"] == ref[0]["lo"]).all() and (gb["votes"] == ref[0]["votes"]).all() and (par.cpu().numpy() == ref[1]).all()
    # new content in the same hit buffer: the replayed graph reads it
    ev2 = g.make_event(rig1.ch, 77, n_noise=20)
    assert ev2.n_hits == ev.n_hits
    hd.copy_(ctx.to_device(b.hits_of(ev2.wire, ev2.drift)))
    ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k, boxes=boxes, params=par)
    ctx.synchronize()
    ob, opar = o.refine(rig1.owires, o.hits_of(ev2.wire, ev2.drift), rig1.oparams, LO, HI, cfg.grid, 5, cfg.k)
    _assert_boxes_equal(b.boxes_to_numpy(boxes, (5, cfg.k)), ob)
    # a different call in between (grows scratch, changes the key), then back
    ctx.ia_vote(hd, ev.n_hits, LO, HI, (12,) * 5)
    ctx.ia_refine(hd, ev.n_hits, LO, HI, (6,) * 5, 3, 4)
    for _ in range(3):
        ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k, boxes=boxes, params=par)
    ctx.synchronize()
    _assert_boxes_equal(b.boxes_to_numpy(boxes, (5, cfg.k)), ob)
    assert (par.cpu().numpy() == opar).all()


# ---- round 2: the tracer itself, the FP32 filter band, edge cases found in review ---------------------------------

def test_tracer_rejects_planted_errors(rig1):
    """G25 tracer (gpu_common.trace_mismatches): a vote that differs for a hit which is NOT on a knife edge must fail, and so
    must per-hit votes that do not add up to the accumulator."""
    from gpu_common import trace_mismatches
    ev = g.make_event(rig1.ch, 21, n_noise=5)
    hd, oh = rig1.hits(ev.wire, ev.drift)
    drift_bad = ev.drift.copy()
    drift_bad[3] += 0.2                                  # one genuine hit mis-measured on the GPU side only
    hd_bad, _ = rig1.hits(ev.wire, drift_bad)
    par = np.array(ev.track.params)
    half = (HI - LO) / 256
    lo, hi = par - half, par + half
    dims = (8, 8, 8, 8, 8)
    vg_bad = rig1.ctx.ia_vote(hd_bad, ev.n_hits, lo, hi, dims).cpu().numpy()
    vg = rig1.ctx.ia_vote(hd, ev.n_hits, lo, hi, dims).cpu().numpy()
    vo = o.vote(rig1.owires, oh, rig1.oparams, lo, hi, dims)
    bad = np.nonzero(vg_bad != vo)[0]
    assert len(bad) > 10
    blo, bhi = o.cell_boxes(lo, hi, dims, bad[:20])
    with pytest.raises(AssertionError, match="unexplained vote mismatch"):
        trace_mismatches(rig1, hd_bad, oh, blo, bhi, vg_bad[bad[:20]], vo[bad[:20]])
    # a wrong count on cells whose per-hit votes all agree
    good = np.nonzero(vg == vo)[0][:5]
    blo, bhi = o.cell_boxes(lo, hi, dims, good)
    assert trace_mismatches(rig1, hd, oh, blo, bhi, vg[good], vo[good]) == 0
    with pytest.raises(AssertionError, match="do not add up"):
        trace_mismatches(rig1, hd, oh, blo, bhi, vg[good] + 1, vo[good])


@pytest.mark.parametrize("precision", [64, 32])
def test_fast_form_stays_within_the_filter_band_of_the_general_form(precision):
    """The sign-specialised form and the general form enclose the same f with different roundings.  Where it matters - at
    an endpoint of f close to zero, where the residual's scale is R_Ax^2 - they must agree to a few ulps of that scale:
    the FP32 path re-takes every decision with an endpoint within 8 ulps of zero (Filter in ia_fast.cuh) in the general
    form, so a difference of more than half of that would let the two forms disagree unnoticed.  (Far from zero the two
    differ by ulps of the larger of R_Ax^2 and (R + d_Ax)^2, which decides nothing.)"""
    rng = np.random.default_rng(77)
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        eps = 2.0 ** -52 if precision == 64 else 2.0 ** -23
        zone = 256 * eps if precision == 32 else 2.0 ** -20           # "close to zero", relative to the scale
        n_fast = n_near = 0
        worst = 0.0
        for lg in range(3, 13):
            for seed in range(3):
                ev = g.make_event(rig.ch, 300 + seed, n_noise=10)
                hd, oh = rig.hits(ev.wire, ev.drift)
                par = np.array(ev.track.params)
                half = (HI - LO) * 2.0 ** -lg / 2
                c = par + rng.uniform(-1, 1, (4000, 5)) * half * 3     # around the truth: f of the genuine hits changes sign
                blo, bhi = c - half, c + half
                blo[:, 2] = np.maximum(blo[:, 2], 20.0)
                bhi[(blo[:, 4] < 0) & (bhi[:, 4] > 0), 4] = 0.0
                lo_d, hi_d = rig.dev(blo), rig.dev(bhi)
                rg = rig.ctx.ia_residual(hd, len(oh), lo_d, hi_d).cpu().numpy()
                rf = rig.ctx.ia_residual_fast(hd, len(oh), lo_d, hi_d).cpu().numpy()
                fast = rf[..., 3] == 0
                n_fast += int(fast.sum())
                assert (rg[..., 3][fast] == 0).all()
                gen = rf[..., 3] == 2                                  # entries that take the general form inside the fast kernel
                assert (rf[..., :2][gen] == rg[..., :2][gen]).all()
                q = rf[..., 2]
                for k in (0, 1):
                    near = fast & (np.minimum(np.abs(rf[..., k]), np.abs(rg[..., k])) < zone * q)
                    n_near += int(near.sum())
                    if near.any():
                        worst = max(worst, float((np.abs(rf[..., k] - rg[..., k])[near] / (eps * q[near])).max()))
        assert n_fast > 1_000_000 and (n_near > 5000 or precision == 64)
        assert worst <= (4.0 if precision == 32 else 16.0), worst
    finally:
        rig.close()


def test_refine_with_no_hits(rig1):
    """No hits at all: every cell has 0 votes, the kept boxes are the first K by index at every level (no division by the
    hit count anywhere in the launch arithmetic)."""
    grid, levels, k = (4, 4, 4, 4, 4), 3, 4
    boxes, par = rig1.ctx.ia_refine(None, 0, LO, HI, grid, levels, k)
    rig1.ctx.synchronize()
    gb = b.boxes_to_numpy(boxes, (levels, k))
    ob, opar = o.refine(rig1.owires, o.hits_of([], []), rig1.oparams, LO, HI, grid, levels, k)
    _assert_boxes_equal(gb, ob)
    assert (gb["votes"] == 0).all() and (par.cpu().numpy() == opar).all()
    # a batch whose events are all empty, sign-specialised and general children kernels
    off = np.zeros(4, np.int32)
    for flags in (0, b.FLAG_GENERAL):
        rig1.ctx.ia_set_params(g.TOL, flags=flags)
        boxes, par = rig1.ctx.ia_refine_batch(None, rig1.dev(off), 3, 0, LO, HI, grid, levels, k)
        rig1.ctx.synchronize()
        gb = b.boxes_to_numpy(boxes, (3, levels, k))
        for e in range(3):
            _assert_boxes_equal(gb[e], ob)
    rig1.ctx.ia_set_params(g.TOL)


def test_many_hits_need_more_than_48k_of_shared_memory(rig1):
    """600 hits per event: the explicit-box kernel and the general children kernel stage 120 B per hit (72 KB) in dynamic
    shared memory, beyond the 48 KB a kernel gets without opting in."""
    rng = np.random.default_rng(5)
    n_hits = 600
    wire = rng.integers(0, rig1.ch.n_wires, n_hits).astype(np.int32)
    drift = rng.uniform(0.0, 1.5, n_hits)
    hd, oh = rig1.hits(wire, drift)
    blo, bhi = _random_boxes(rng, 300, 2, 9)
    vg = rig1.ctx.ia_vote_boxes(hd, n_hits, rig1.dev(blo), rig1.dev(bhi))
    rig1.ctx.synchronize()
    vo = o.vote_boxes(rig1.owires, oh, rig1.oparams, blo, bhi)
    # 300 boxes x 600 hits = 180,000 decisions: up to three traced knife-edge boxes allowed
    compare_votes(rig1, hd, oh, vg.cpu().numpy(), vo, lambda idx: (blo[idx], bhi[idx]), min_equal=0.99, kind="boxes")
    # general-form refinement (IA_FLAG_GENERAL) of 300 events x 420 hits: one hit split per event, all hits in one block
    n_events, mh = 300, 420
    wire = rng.integers(0, rig1.ch.n_wires, n_events * mh).astype(np.int32)
    drift = rng.uniform(0.0, 1.5, n_events * mh)
    off = (np.arange(n_events + 1) * mh).astype(np.int32)
    hd, oh = rig1.hits(wire, drift)
    grid, levels, k = (3, 3, 3, 2, 2), 2, 4
    rig1.ctx.ia_set_params(g.TOL, flags=b.FLAG_GENERAL)
    try:
        boxes, par = rig1.ctx.ia_refine_batch(hd, rig1.dev(off), n_events, mh, LO, HI, grid, levels, k)
        rig1.ctx.synchronize()
    finally:
        rig1.ctx.ia_set_params(g.TOL)
    gb = b.boxes_to_numpy(boxes, (n_events, levels, k))
    ob, opar = o.refine_batch(rig1.owires, oh, off, rig1.oparams, LO, HI, grid, levels, k)
    _assert_boxes_equal(gb, ob)


def test_refine_graph_is_really_replayed_on_a_capturable_stream():
    """The legacy default stream cannot be captured, so a Context made on it always launches directly (replays stay 0);
    on an explicit stream the third identical call on is one cudaGraphLaunch - and gives the same boxes."""
    import torch
    cfg = g.config(2)
    ev = cfg.events[0]
    ctx = b.Context(0, stream=torch.cuda.Stream())
    try:
        ctx.ia_load_geometry(b.wires_of(cfg.chamber))
        ctx.ia_set_params(g.TOL)
        hd = ctx.to_device(b.hits_of(ev.wire, ev.drift))
        torch.cuda.synchronize()
        boxes, par = ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k)
        ctx.synchronize()
        ref = b.boxes_to_numpy(boxes, (5, cfg.k)).copy()
        assert ctx.ia_graph_replays() == 0
        for i in range(4):
            l0 = ctx.ia_launch_count()
            ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 5, cfg.k, boxes=boxes, params=par)
            ctx.synchronize()
            assert ctx.ia_launch_count() > l0
            gb = b.boxes_to_numpy(boxes, (5, cfg.k))
            assert (gb["lo"] == ref["lo"]).all() and (gb["hi"] == ref["hi"]).all() and (gb["votes"] == ref["votes"]).all()
        assert ctx.ia_graph_replays() == 4, ctx.ia_graph_replays()        # the second call captures and launches the graph, 3-5 replay it
        ob, _ = o.refine(o.wires_of(cfg.chamber), o.hits_of(ev.wire, ev.drift), o.make_params(g.TOL), LO, HI, cfg.grid, 5, cfg.k)
        _assert_boxes_equal(ref, ob)
    finally:
        ctx.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_prefilter_gives_identical_votes(precision):
    """IA_FLAG_PREFILTER: hits that a crude enclosure (magnitude bounds over a whole z0 tile) excludes for every lane of a warp
    are skipped.  A wider enclosure that excludes 0 implies the fine one does, so the accumulator must be identical bit for
    bit to the exhaustive kernel's - on a fine grid (where most hits are skipped), a coarse one, ragged shapes, a window
    around the truth (where few are), an odd lambda grid, and with the reference plane and point off zero."""
    import torch
    for ref in ((0.0, 0.0, 0.0), (1.5, -2.0, 3.0)):
        rig = Rig(g.chamber_c1(), precision=precision, x_ref=ref[0], y_ref=ref[1], z_ref=ref[2])
        try:
            ev = g.make_event(rig.ch, 35, n_noise=10)
            hd, oh = rig.hits(ev.wire, ev.drift)
            par = np.array(ev.track.params)
            half = (HI - LO) / 128
            grids = [(LO, HI, (24,) * 5), (LO, HI, (8,) * 5), (LO, HI, (5, 4, 10, 37, 12)), (LO, HI, (3, 3, 6, 20, 7)),
                     (par - half, par + half, (8, 8, 8, 8, 8)), (LO, HI, (40, 40, 8, 4, 8))]
            for lo, hi, dims in grids:
                out = []
                for flags in (0, 64):
                    rig.ctx.ia_set_params(g.TOL, ref[0], ref[1], ref[2], precision, flags)
                    out.append(rig.ctx.ia_vote(hd, ev.n_hits, lo, hi, dims))
                rig.ctx.synchronize()
                a, c = out[0].cpu().numpy(), out[1].cpu().numpy()
                assert (a == c).all(), (precision, ref, dims, int((a != c).sum()), np.nonzero(a != c)[0][:10], a[a != c][:10], c[a != c][:10])
                assert a.max() > 0
        finally:
            rig.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_slab_votes_tile_the_accumulator_and_key_lists_merge_to_the_same_topk(precision):
    """SURVEY 8(e), one event on several GPUs: the slabs of ia_vote_slab (2, 3, 5 and 8 "ranks", run one after the other on
    this GPU - no rank waits for another) concatenate to ia_vote's accumulator count for count, the merged key lists of
    ia_topk_keys give ia_topk's result on the whole accumulator, and that is the oracle's top-K of the oracle's votes."""
    import torch
    from paper_2401_04576_b200 import shard
    rig = Rig(g.chamber_c1(), precision=precision)
    try:
        ev = g.make_event(rig.ch, 11, n_noise=20)
        hd, oh = rig.hits(ev.wire, ev.drift)
        for dims, k in (((12, 10, 12, 12, 12), 10), ((5, 7, 6, 9, 3), 32), ((3, 4, 8, 8, 8), 16)):
            full = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            idx_f, v_f = rig.ctx.ia_topk(full, k)
            rig.ctx.synchronize()
            col = int(np.prod(dims[1:]))
            for world in (2, 3, 5, 8):
                slabs, lists = [], []
                for rank in range(world):
                    b0, e0 = shard.slab_range(dims[0], rank, world)
                    if e0 > b0:
                        vs = rig.ctx.ia_vote_slab(hd, ev.n_hits, LO, HI, dims, b0, e0)
                        lists.append(rig.ctx.ia_topk_keys(vs, min(k, (e0 - b0) * col), index_base=b0 * col))
                        slabs.append(vs)
                    else:
                        lists.append(torch.zeros(32, dtype=torch.int64, device="cuda"))
                rig.ctx.synchronize()
                assert torch.equal(torch.cat(slabs).view(torch.int16), full.view(torch.int16)), (dims, world)
                idx_m, v_m = rig.ctx.ia_merge_keys(torch.cat(lists), world, k)
                rig.ctx.synchronize()
                assert torch.equal(idx_m, idx_f) and torch.equal(v_m.view(torch.int16), v_f.view(torch.int16)), (dims, world)
            # the single-process form of the whole split path
            idx_s, v_s, _ = shard.split_vote_topk(rig.ctx, hd, ev.n_hits, LO, HI, dims, k)
            rig.ctx.synchronize()
            assert torch.equal(idx_s, idx_f)
            vo = o.vote(rig.owires, oh, rig.oparams, LO, HI, dims)
            eidx, evv = o.topk(full.cpu().numpy(), k)
            assert (idx_f.cpu().numpy() == eidx).all() and (v_f.cpu().numpy() == evv).all()
            assert (full.cpu().numpy() == vo).mean() >= 0.9999
        # errors: a range outside the axis
        with pytest.raises(b.IaError):
            rig.ctx.ia_vote_slab(hd, ev.n_hits, LO, HI, (4, 4, 4, 4, 4), 2, 5)
    finally:
        rig.close()


def test_outputs_stay_inside_their_buffers(rig1):
    """compute-sanitizer is closed on this GPU pool, so: every caller-provided output is a window inside a larger buffer
    of canary bytes, on shapes chosen to end in partial warps, partial tiles and odd strides; after the calls the canaries
    on both sides are intact and the window equals what the same call writes into a buffer of its own."""
    import torch
    ctx = rig1.ctx
    ev = g.make_event(rig1.ch, 5, n_noise=7)
    hd, _ = rig1.hits(ev.wire, ev.drift)
    GUARD = 4096

    def window(nbytes, dtype):
        buf = torch.full((nbytes + 2 * GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
        return buf, buf[GUARD:GUARD + nbytes].view(dtype)

    def intact(buf, nbytes):
        return bool((buf[:GUARD] == 0xA5).all()) and bool((buf[GUARD + nbytes:] == 0xA5).all())

    for prec in (64, 32):
        ctx.ia_set_params(g.TOL, precision=prec)
        # dense vote: ragged grids (partial pair tiles, partial z0 tiles, odd lambda count), the general kernel, a slab
        for dims, flags in (((3, 2, 7, 5, 9), 0), ((2, 3, 33, 17, 10), 0), ((2, 2, 5, 19, 3), 1), ((1, 1, 1, 1, 1), 0)):
            ctx.ia_set_params(g.TOL, precision=prec, flags=flags)
            n = int(np.prod(dims))
            buf, w = window(2 * n, torch.uint16)
            ctx.ia_vote(hd, ev.n_hits, LO, HI, dims, votes_out=w)
            ref = ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            ctx.synchronize()
            assert intact(buf, 2 * n) and torch.equal(w.view(torch.int16), ref.view(torch.int16)), (prec, dims, flags)
        ctx.ia_set_params(g.TOL, precision=prec)
        dims = (5, 3, 9, 7, 4)
        col = int(np.prod(dims[1:]))
        buf, w = window(2 * 2 * col, torch.uint16)
        ctx.ia_vote_slab(hd, ev.n_hits, LO, HI, dims, 2, 4, votes_out=w)
        full = ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
        ctx.synchronize()
        assert intact(buf, 4 * col) and torch.equal(w.view(torch.int16), full[2 * col:4 * col].view(torch.int16))
        # explicit boxes: a count that is not a multiple of the block
        nb = 131
        blo = np.tile(LO, (nb, 1)) + np.linspace(0, 1, nb)[:, None] * 0.3 * (HI - LO)
        bhi = blo + 0.1 * (HI - LO)
        buf, w = window(2 * nb, torch.uint16)
        ctx.ia_vote_boxes(hd, ev.n_hits, rig1.dev(blo), rig1.dev(bhi), votes_out=w)
        ref = ctx.ia_vote_boxes(hd, ev.n_hits, rig1.dev(blo), rig1.dev(bhi))
        ctx.synchronize()
        assert intact(buf, 2 * nb) and torch.equal(w.view(torch.int16), ref.view(torch.int16))
        # refinement: boxes and parameters, single event and a batch with an empty event, K not a power of two
        for levels, k in ((3, 5), (4, 16)):
            nbx = levels * k * b.BOX_DT.itemsize
            bb, wb = window(nbx, torch.uint8)
            pb, wp = window(8 * b.IA_N_PARAMS, torch.float64)
            ctx.ia_refine(hd, ev.n_hits, LO, HI, (4, 4, 4, 4, 4), levels, k, boxes=wb, params=wp)
            rb_, rp_ = ctx.ia_refine(hd, ev.n_hits, LO, HI, (4, 4, 4, 4, 4), levels, k)
            ctx.synchronize()
            assert intact(bb, nbx) and intact(pb, 8 * b.IA_N_PARAMS) and torch.equal(wb, rb_) and torch.equal(wp, rp_)
        evs = [g.make_event(rig1.ch, 40 + e, n_noise=3) for e in range(3)]
        wire = np.concatenate([evs[0].wire, evs[2].wire]); drift = np.concatenate([evs[0].drift, evs[2].drift])
        off = np.array([0, evs[0].n_hits, evs[0].n_hits, evs[0].n_hits + evs[2].n_hits], np.int32)
        hb, _ = rig1.hits(wire, drift)
        levels, k = 3, 7
        nbx = 3 * levels * k * b.BOX_DT.itemsize
        bb, wb = window(nbx, torch.uint8)
        pb, wp = window(3 * 8 * b.IA_N_PARAMS, torch.float64)
        mh = int(max(evs[0].n_hits, evs[2].n_hits))
        ctx.ia_refine_batch(hb, rig1.dev(off), 3, mh, LO, HI, (4, 4, 4, 4, 4), levels, k, boxes=wb, params=wp)
        rb_, rp_ = ctx.ia_refine_batch(hb, rig1.dev(off), 3, mh, LO, HI, (4, 4, 4, 4, 4), levels, k)
        ctx.synchronize()
        assert intact(bb, nbx) and intact(pb, 3 * 8 * b.IA_N_PARAMS) and torch.equal(wb, rb_) and torch.equal(wp, rp_)
    # paper mode (double): two accumulators of an odd-shaped grid
    ctx.ia_set_params(g.TOL)
    xc, yc, R, z0, lam = ev.track.params
    P = R * (1.0 + lam * lam) ** 0.5
    d4 = (7, 5, 9, 3)
    n4 = int(np.prod(d4))
    buf, w = window(2 * 2 * n4, torch.uint16)
    ctx.ia_vote_paper(hd, ev.n_hits, P, LO[:4], HI[:4], d4, votes_out=w)
    ref = ctx.ia_vote_paper(hd, ev.n_hits, P, LO[:4], HI[:4], d4)
    ctx.synchronize()
    assert intact(buf, 4 * n4) and torch.equal(w.view(torch.int16), ref.reshape(-1).view(torch.int16))


def test_programmatic_dependent_launch_changes_nothing(rig1):
    """IA_FLAG_NO_PDL launches the chain without the programmatic-dependent-launch attribute: same boxes and parameters,
    replayed as a graph or not (IA_FLAG_NO_GRAPH), and the same dense votes and top-K."""
    import torch
    cfg = g.config(2)
    ev = cfg.events[0]
    hd, _ = rig1.hits(ev.wire, ev.drift)
    ctx = rig1.ctx
    ref = None
    for flags in (0, b.FLAG_NO_PDL, b.FLAG_NO_GRAPH, b.FLAG_NO_PDL | b.FLAG_NO_GRAPH):
        ctx.ia_set_params(g.TOL, flags=flags)
        for _ in range(3):                                   # third call: the graph replay where it applies
            boxes, par = ctx.ia_refine(hd, ev.n_hits, LO, HI, cfg.grid, 6, cfg.k)
        v = ctx.ia_vote(hd, ev.n_hits, LO, HI, (6, 5, 9, 7, 4))
        idx, vv = ctx.ia_topk(v, 10)
        ctx.synchronize()
        got = (boxes.clone(), par.clone(), v.view(torch.int16).clone(), idx.clone())
        if ref is None:
            ref = got
        else:
            assert all(torch.equal(a, c) for a, c in zip(ref, got)), flags
    ctx.ia_set_params(g.TOL)
