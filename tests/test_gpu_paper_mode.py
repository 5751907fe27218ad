"""-m gpu parity of ia_vote_paper against the oracle's paper mode.

Both sides evaluate d_Ax in round-to-nearest double with the same operations in the same order; they
differ only through sin, cos and atan2 (glibc against CUDA / the kernel's own Taylor forms: a few ulps of
d_Ax).  Bar: every voxel of both accumulators equal in >= 99.99 %, and every mismatch traced to a
(voxel, hit, lambda sign, drift sign) whose oracle enclosure of condition (4) has an endpoint within
1e-12 (relative to the residual's scale) of zero.
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import binding as b
from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

from gpu_common import Rig

pytestmark = pytest.mark.gpu

LO4, HI4 = np.array(g.BOX_LO[:4]), np.array(g.BOX_HI[:4])


def _momentum_radius(ev):
    xc, yc, R, z0, lam = ev.track.params
    return R * np.sqrt(1.0 + lam * lam)


def _compare(rig, ev, P, lo, hi, dims, tol):
    hd, oh = rig.hits(ev.wire, ev.drift)
    rig.ctx.ia_set_params(tol)
    vg = rig.ctx.ia_vote_paper(hd, ev.n_hits, P, lo, hi, dims)
    rig.ctx.synchronize()
    vg = vg.cpu().numpy()
    op = o.make_params(tol)
    vo = o.vote_paper(rig.owires, oh, op, P, lo, hi, dims)
    assert vg.shape == vo.shape
    bad = np.argwhere(vg != vo)
    n = vo.size
    assert len(bad) <= n * 1e-4, (len(bad), n)
    # trace every mismatch (G25 applied to condition (4))
    if len(bad):
        cells = np.unique(bad[:, 1])
        blo, bhi = o.cell_boxes4(lo, hi, dims, cells)
        r = o.residual_paper(rig.owires, oh, op, P, blo, bhi)
        for i in range(len(cells)):
            knife = (r[i, ..., 3] > 0) & (np.minimum(np.abs(r[i, ..., 0]), np.abs(r[i, ..., 1])) <= 1e-12 * r[i, ..., 2])
            assert knife.any(), f"unexplained paper-mode mismatch in voxel {cells[i]}"
    return vg, vo, len(bad)


@pytest.mark.parametrize("tol", [g.TOL, 0.0])
def test_paper_mode_c1_event_every_voxel(tol):
    """20-layer chamber, 1 track + 20 noise hits; a Table-1-shaped coarse grid (L100-106), every voxel."""
    rig = Rig(g.chamber_c1())
    try:
        ev = g.make_event(rig.ch, 1, n_noise=20)
        P = _momentum_radius(ev)
        vg, vo, nbad = _compare(rig, ev, P, LO4, HI4, (25, 25, 20, 10), tol)
        assert vo.max() > 0
        rm_gt = vo.reshape(2, 25, 25, 20, 10)
        assert rm_gt.shape[0] == 2
    finally:
        rig.close()


def test_paper_mode_ragged_window_and_negative_lambda():
    """ragged dims spanning several blocks and a partial one; a window grid around the truth (Table 1, iteration
    3 shape) where the truth voxel must collect the genuine hits in the accumulator of the true lambda sign."""
    rig = Rig(g.chamber_c1())
    try:
        seen = set()
        for seed in (11, 12, 13, 14, 15, 16):
            ev = g.make_event(rig.ch, seed, n_noise=8)
            xc, yc, R, z0, lam = ev.track.params
            if abs(lam) < 0.1:
                continue
            seen.add(lam > 0)
            P = _momentum_radius(ev)
            c = np.array([xc, yc, R, z0])
            hw = np.array([2.5, 2.5, 2.5, 4.0])
            dims = (9, 7, 13, 5)
            vg, vo, _ = _compare(rig, ev, P, c - hw, c + hw, dims, g.TOL)
            good = 0 if lam > 0 else 1
            centre = (((4 * 7 + 3) * 13 + 6) * 5 + 2)
            genuine = int((~ev.is_noise & ~ev.clipped).sum())
            assert vg[good, centre] >= genuine - 1, (seed, vg[:, centre], genuine)
            assert vg[good].max() >= vg[1 - good].max()
        assert seen == {True, False}
    finally:
        rig.close()


def test_paper_mode_degenerate_and_errors():
    rig = Rig(g.chamber_c0())
    try:
        ev = g.make_event(rig.ch, 0)
        hd, oh = rig.hits(ev.wire, ev.drift)
        P = _momentum_radius(ev)
        # one voxel; a grid whose R range lies entirely above P (no lambda anywhere -> all zero)
        _compare(rig, ev, P, LO4, HI4, (1, 1, 1, 1), g.TOL)
        lo, hi = LO4.copy(), HI4.copy()
        lo[2], hi[2] = P * 1.01, P * 1.5
        v = rig.ctx.ia_vote_paper(hd, ev.n_hits, P, lo, hi, (3, 3, 4, 2))
        rig.ctx.synchronize()
        assert int(v.cpu().numpy().max()) == 0
        # no hits: zero votes
        v = rig.ctx.ia_vote_paper(None, 0, P, LO4, HI4, (2, 2, 2, 2))
        rig.ctx.synchronize()
        assert int(v.cpu().numpy().max()) == 0
        with pytest.raises(b.IaError) as ei:
            rig.ctx.ia_vote_paper(hd, ev.n_hits, -1.0, LO4, HI4, (2, 2, 2, 2))
        assert ei.value.code == -1
        lo = LO4.copy()
        lo[2] = 0.0
        with pytest.raises(b.IaError) as ei:
            rig.ctx.ia_vote_paper(hd, ev.n_hits, P, lo, HI4, (2, 2, 2, 2))
        assert ei.value.code == -3
    finally:
        rig.close()


# ---- pieces of the paper's iteration scheme ---------------------------------------------------
def _fit_to_host(t):
    return np.frombuffer(t.cpu().numpy().tobytes(), dtype=b.FIT_DT)[0]


def test_f2_disk_filter_hit_mask_selection_and_hit_finding():
    """ia_vote_paper with a hit mask and the disk pre-filter, ia_select_max_paper and ia_find_hits_paper against the
    oracle: accumulators equal (>= 99.99 %, traced), the selection bit-identical (integer sums), flags identical."""
    rig = Rig(g.chamber_c1())
    try:
        for seed, dims in ((21, (20, 20, 16, 8)), (22, (13, 11, 9, 7)), (23, (30, 30, 10, 4))):
            ev = g.make_event(rig.ch, seed, n_noise=15)
            P = _momentum_radius(ev)
            hd, oh = rig.hits(ev.wire, ev.drift)
            mask = (np.arange(ev.n_hits) % 4 != 1).astype(np.uint8)
            rig.ctx.ia_set_params(g.TOL)
            vg = rig.ctx.ia_vote_paper(hd, ev.n_hits, P, LO4, HI4, dims, hit_mask_dev=rig.dev(mask), r_disk=10.0)
            fit_dev = rig.ctx.ia_select_max_paper(vg.view(-1), P, LO4, HI4, dims)
            flags = rig.ctx.ia_find_hits_paper(hd, ev.n_hits, P, fit_dev, 5.0)
            rig.ctx.synchronize()
            vg_h = vg.cpu().numpy()
            op = o.make_params(g.TOL)
            vo = o.vote_paper(rig.owires, oh, op, P, LO4, HI4, dims, hit_mask=mask, r_disk=10.0)
            assert (vg_h != vo).sum() <= vo.size * 1e-4
            keep = o.disk_filter(LO4, HI4, dims, 10.0)
            assert (vg_h[:, keep == 0] == 0).all() and 0 < keep.sum() < keep.size
            # selection: defined on the accumulators it is given -> compare on the GPU's own accumulators
            fo = o.select_max_paper(vg_h, LO4, HI4, dims, P)
            fg = _fit_to_host(fit_dev)
            assert list(fg["value"]) == list(fo.value) and list(fg["error"]) == list(fo.error)
            assert fg["vmax"] == fo.vmax and fg["n_sel"] == fo.n_sel and fg["lambda_sign"] == fo.lambda_sign
            assert fg["lam"] == fo.lam
            # hit finding on value -/+ 5 error (rn, unfused - the same two operations as the kernel)
            val, err = np.array(fo.value), np.array(fo.error)
            lo, hi = val - 5.0 * err, val + 5.0 * err
            fl_o = o.find_hits_paper(rig.owires, oh, op, P, fo.lambda_sign, lo, hi)
            assert (flags.cpu().numpy() == fl_o).all()
            assert fl_o.sum() > 0
    finally:
        rig.close()


def test_f2_selection_special_cases_on_device():
    """hand-made accumulators: single voxel, block, ties between the accumulators, all-equal counts (every voxel
    selected: the centre of the grid, half its size)."""
    import torch
    rig = Rig(g.chamber_c0())
    try:
        dims = (10, 8, 6, 4)
        lo, hi = np.array([-100.0, -80.0, 60.0, -8.0]), np.array([100.0, 80.0, 120.0, 8.0])
        n = int(np.prod(dims))
        rng = np.random.default_rng(9)
        cases = []
        v = np.full((2, n), 3, np.uint16); v[0, 777] = 9; cases.append(v)
        v = np.full((2, n), 3, np.uint16); v[1, 100:140] = 5; cases.append(v)
        v = np.full((2, n), 2, np.uint16); cases.append(v)
        v = rng.integers(0, 4, (2, n)).astype(np.uint16); cases.append(v)
        v = rng.integers(0, 30, (2, n)).astype(np.uint16); v[1, 5] = 40; v[0, 6] = 40; cases.append(v)
        for v in cases:
            fit_dev = rig.ctx.ia_select_max_paper(torch.from_numpy(v.view(np.int16).copy()).view(torch.uint16).cuda().view(-1),
                                                  150.0, lo, hi, dims)
            rig.ctx.synchronize()
            fg, fo = _fit_to_host(fit_dev), o.select_max_paper(v, lo, hi, dims, 150.0)
            assert list(fg["value"]) == list(fo.value) and list(fg["error"]) == list(fo.error)
            assert (fg["vmax"], fg["n_sel"], fg["lambda_sign"], fg["lam"]) == (fo.vmax, fo.n_sel, fo.lambda_sign, fo.lam)
    finally:
        rig.close()


# ---- the iteration scheme as one call (f2) on the paper-shaped workload (f4) ------------------------------------------
PLO, PHI = np.array(g.PAPER_BOX_LO), np.array(g.PAPER_BOX_HI)


def _passes(spec, move_ref=False):
    ps = np.zeros(len(spec), b.PASS_DT)
    ps["move_ref"][1:] = 1 if move_ref else 0          # L98: every pass but the first is voted with the moved reference point
    for i, s in enumerate(spec):
        if s[0] == "grid":
            ps[i]["lo"], ps[i]["hi"], ps[i]["dims"], ps[i]["windowed"] = s[1], s[2], s[3], 0
        else:
            ps[i]["lo"], ps[i]["hi"], ps[i]["dims"], ps[i]["windowed"] = s[1], s[1], s[2], 1
    return ps


def _fits_to_host(t, n_passes):
    return np.frombuffer(t.cpu().numpy().tobytes(), dtype=b.FIT_DT).reshape(n_passes, 2)


def test_track_paper_matches_the_oracle_chain():
    """ia_track_paper against orc_track_paper on reduced grids (the oracle needs seconds per pass): every fit of every
    pass and both chains identical, same final sign.  Tracks of more than half a turn (IA_FLAG_FULL_TURN)."""
    ch = g.chamber_paper()
    rig = Rig(ch)
    try:
        spec = [("grid", PLO, PHI, (24, 24, 16, 10)), ("grid", PLO, PHI, (36, 36, 16, 10)),
                ("window", (3.0, 3.0, 2.0, 30.0), (20, 20, 16, 10))]
        # fixed reference point, then the reference point of L98 (reading F2d') on tracks from the origin and from (5, 0) cm
        for seed, move, vertex in ((300, False, (0.0, 0.0)), (301, False, (0.0, 0.0)), (302, False, (0.0, 0.0)),
                                   (300, True, (0.0, 0.0)), (301, True, (0.0, 0.0)), (303, True, (5.0, 0.0)), (304, True, (0.0, 5.0))):
            ev = g.make_event_paper(ch, seed, n_noise=3, vertex=vertex)
            hd, oh = rig.hits(ev.wire, ev.drift)
            rig.ctx.ia_set_params(0.01, flags=b.FLAG_FULL_TURN)
            fits_dev, sign_dev = rig.ctx.ia_track_paper(hd, ev.n_hits, g.PAPER_P, _passes(spec, move), r_disk=10.0, factor=5.0)
            rig.ctx.synchronize()
            fg = _fits_to_host(fits_dev, len(spec))
            fo, so = o.track_paper(rig.owires, oh, o.make_params(0.01, flags=8), g.PAPER_P, 10.0, 5.0, o.make_passes(spec, move))
            assert int(sign_dev.cpu().numpy()[0]) == so
            for name in ("lambda_sign", "x_ref", "y_ref"):
                assert (fg[name] == fo[name]).all(), (seed, move, name, fg[name], fo[name])
            for name in ("vmax", "n_sel"):
                # identical wherever the two sides vote the same grid.  The window of a pass whose reference point moved
                # is centred on a z0 transported with atan2 (CUDA's against glibc's): where that centre differs in its
                # last bits the voxel edges do too, and a knife-edge vote may flip - allowed there only, by one vote
                same_grid = fg["z0_centre"] == fo["z0_centre"]
                differ = fg[name] != fo[name]
                assert not (differ & same_grid).any(), (seed, move, name, fg[name], fo[name])
                assert not differ[:2].any(), (seed, move, name, fg[name], fo[name])
            assert (np.abs(fg["vmax"].astype(np.int64) - fo["vmax"]) <= 1).all()
            assert np.allclose(fg["z0_centre"], fo["z0_centre"], rtol=0, atol=1e-9)      # transported with atan2: to rounding
            for name in ("value", "error", "lam"):
                # the global passes bit for bit; the window after a moved reference point is centred on a z0 transported
                # with atan2 (CUDA's against glibc's: an ulp), so its grid - and with it the fit - agrees to rounding
                assert (fg[name][:2] == fo[name][:2]).all(), (seed, move, name, fg[name], fo[name])
                if move:
                    assert np.allclose(fg[name][2], fo[name][2], rtol=0, atol=1e-9), (seed, name, fg[name][2], fo[name][2])
                else:
                    assert (fg[name][2] == fo[name][2]).all(), (seed, name, fg[name][2], fo[name][2])
            assert (fg["x_ref"][0] == 0.0).all() and (fg["y_ref"][0] == 0.0).all()
            if move:
                assert (np.hypot(fg["x_ref"][1:], fg["y_ref"][1:]) > 40.0).all()      # on a wire of the chamber (r >= 49.6 cm)
    finally:
        rig.close()


def test_table1_first_pass_every_voxel():
    """The first pass of the paper's scheme at the size Table 1 gives it (L100-106: 50 x 50 x 40 x 20 voxels on the global
    box), on a paper-shaped event with the disk pre-filter (3a,b) and tracks of up to one turn: both lambda-sign
    accumulators of ia_vote_paper against orc_vote_paper, voxel for voxel (the reduced grids of the chain test above
    keep the oracle's time down; this is the one pass at full size).  Then the selection on both sides."""
    ch = g.chamber_paper()
    rig = Rig(ch)
    try:
        ev = g.make_event_paper(ch, 500)
        hd, oh = rig.hits(ev.wire, ev.drift)
        dims = (50, 50, 40, 20)
        rig.ctx.ia_set_params(0.0, flags=b.FLAG_FULL_TURN)
        vg_dev = rig.ctx.ia_vote_paper(hd, ev.n_hits, g.PAPER_P, PLO, PHI, dims, r_disk=10.0)
        fit_dev = rig.ctx.ia_select_max_paper(vg_dev.view(-1), g.PAPER_P, PLO, PHI, dims)
        rig.ctx.synchronize()
        vg = vg_dev.cpu().numpy()
        op = o.make_params(0.0, flags=8)
        vo = o.vote_paper(rig.owires, oh, op, g.PAPER_P, PLO, PHI, dims, r_disk=10.0)
        assert vg.shape == vo.shape == (2, 2_000_000) and vo.max() >= 5
        bad = np.argwhere(vg != vo)
        assert len(bad) <= vo.size * 1e-4, len(bad)
        if len(bad):
            cells = np.unique(bad[:, 1])
            blo, bhi = o.cell_boxes4(PLO, PHI, dims, cells)
            r = o.residual_paper(rig.owires, oh, op, g.PAPER_P, blo, bhi)
            for i in range(len(cells)):
                knife = (r[i, ..., 3] > 0) & (np.minimum(np.abs(r[i, ..., 0]), np.abs(r[i, ..., 1])) <= 1e-12 * r[i, ..., 2])
                assert knife.any(), f"unexplained paper-mode mismatch in voxel {cells[i]}"
        # the selection is defined on the accumulators it is given: the oracle's on the GPU's own accumulators
        fg, fo = _fit_to_host(fit_dev), o.select_max_paper(vg, PLO, PHI, dims, g.PAPER_P)
        assert list(fg["value"]) == list(fo.value) and list(fg["error"]) == list(fo.error)
        assert (fg["vmax"], fg["n_sel"], fg["lambda_sign"], fg["lam"]) == (fo.vmax, fo.n_sel, fo.lambda_sign, fo.lam)
    finally:
        rig.close()


def test_track_paper_recovers_the_generated_helix():
    """Table 1 of the paper in cm (L100-106): two global passes (voxels 1.8 x 1.8 x 0.375 x 7.5 and 1.0 x 1.0 x 0.375 x 7.5
    cm) and a window of +/-2.5, 2.5, 2.5, 40 cm with voxels 0.1 x 0.1 x 0.1 x 4 cm, on noise-free paper-shaped events
    (L88).  Measured, then asserted loosely: the sign of lambda and the helix within a few final voxels."""
    ch = g.chamber_paper()
    rig = Rig(ch)
    try:
        spec = [("grid", PLO, PHI, (50, 50, 40, 20)), ("grid", PLO, PHI, (90, 90, 40, 20)),
                ("window", (2.5, 2.5, 2.5, 40.0), (50, 50, 50, 20))]
        rig.ctx.ia_set_params(0.0, flags=b.FLAG_FULL_TURN)
        for move, vertex in ((False, (0.0, 0.0)), (True, (0.0, 0.0)), (True, (5.0, 0.0))):
            ok_sign, dev = 0, []
            seeds = range(400, 424)
            for seed in seeds:
                ev = g.make_event_paper(ch, seed, vertex=vertex)
                hd, _ = rig.hits(ev.wire, ev.drift)
                fits_dev, sign_dev = rig.ctx.ia_track_paper(hd, ev.n_hits, g.PAPER_P, _passes(spec, move))
                rig.ctx.synchronize()
                fg = _fits_to_host(fits_dev, 3)
                s = int(sign_dev.cpu().numpy()[0])
                ok_sign += s == (1 if ev.track.lam >= 0 else -1)
                f = fg[2, 0 if s > 0 else 1]
                # z0 of a fit is relative to the reference point of its pass: compare with the generated helix there
                truth = np.array(ev.track.params_at(float(f["x_ref"]), float(f["y_ref"]), unwrap=True)[:4])
                dev.append(np.abs(np.array(f["value"]) - truth))
            dev = np.array(dev)
            assert ok_sign >= len(seeds) - 1, (move, vertex, ok_sign)
            good = (dev[:, :3] < 0.3).all(axis=1) & (dev[:, 3] < 4.0)
            assert good.mean() >= 0.9, (move, vertex, good.mean(), np.median(dev, axis=0))
            assert (np.median(dev, axis=0) < np.array([0.1, 0.1, 0.1, 2.0])).all(), (move, vertex, np.median(dev, axis=0))
    finally:
        rig.close()


def test_f2_selection_when_every_voxel_is_selected():
    """a plateau that holds the whole grid (all counts equal): the centre of the grid and half its size, also on a
    grid of millions of voxels (the reduction aggregates per warp before its atomics)."""
    import torch
    rig = Rig(g.chamber_c0())
    try:
        dims = (64, 64, 32, 16)
        n = int(np.prod(dims))
        v = torch.full((2 * n,), 5, dtype=torch.int16, device="cuda").view(torch.uint16)
        fit_dev = rig.ctx.ia_select_max_paper(v, 300.0, PLO, PHI, dims)
        rig.ctx.synchronize()
        f = _fit_to_host(fit_dev)
        assert f["n_sel"] == n and f["vmax"] == 5 and f["lambda_sign"] == 1
        assert np.allclose(f["value"], 0.5 * (PLO + PHI), rtol=0, atol=1e-9)
        assert np.allclose(f["error"], 0.5 * (PHI - PLO), rtol=0, atol=1e-9)
    finally:
        rig.close()
