"""Pins of the oracle's residual enclosure (steps S1-S8).

P1  identity at the generated truth: with thin intervals, tol=0 and the true drift sign, the
    enclosure sits on zero up to the (unenclosed) series truncation: |sqrt(Q) - sqrt(rad)| <= 1 um.
--  thin enclosures equal the independent numpy point model (tests/pointmodel.py, itself pinned
    to the paper's exact identities in test_eventgen.py) at random, off-truth points.
P5  brute-force sampling on tiny grids: the point model sampled at corners + interior points never
    leaves the enclosure; enclosure width stays within a small factor of the sampled range.
P6  inclusion isotonicity: child box in parent box => enclosure(child) in enclosure(parent).
--  FP32 mode encloses the FP64 enclosure when every scalar input is float-representable.
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

import pointmodel as pm


def _wire_tuple(ch, wid):
    return (ch.x0[wid], ch.y0[wid], ch.sin_phi_s[wid], ch.cos_phi_s[wid], ch.tan_tau[wid])


@pytest.mark.parametrize("chamber", [g.chamber_c0, g.chamber_c1, g.chamber_c4])
def test_p1_identity_at_truth(chamber):
    ch = chamber()
    wires = o.wires_of(ch)
    p = o.make_params(0.0)
    worst = 0.0
    for seed in range(25):
        ev = g.make_event(ch, 500 + seed, smear=0.0)
        par = np.array(ev.track.params)
        hits = o.hits_of(ev.wire, np.abs(ev.d_true))
        r = o.residual(wires, hits, p, par[None], par[None])[0]
        for i in range(ev.n_hits):
            sg = 0 if ev.d_true[i] > 0 else 1
            flo, fhi, scale, decided = r[i, sg]
            assert not decided and flo <= fhi
            RA = np.sqrt(scale)
            # sqrt(Q) - sqrt(rad) = f / (sqrt(Q) + sqrt(rad)) ~ f / (2 RA)
            err_cm = max(abs(flo), abs(fhi)) / (2 * RA)
            worst = max(worst, err_cm)
            assert err_cm <= 1e-4, (seed, i, err_cm)            # 1 um
            assert fhi - flo <= 1e-9 * scale                    # thin stays thin
            # the wrong sign is off by about 2|d|: excluded unless the drift is tiny
            wlo, whi = r[i, 1 - sg][:2]
            if abs(ev.d_true[i]) > 0.01:
                assert wlo > 0 or whi < 0
    assert worst > 0        # the series is an approximation: not identically zero


def test_thin_enclosure_equals_point_model():
    rng = np.random.default_rng(7)
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    for z_ref, xr, yr in ((0.0, 0.0, 0.0), (2.5, 1.0, -3.0)):
        p = o.make_params(0.0, xr, yr, z_ref)
        for _ in range(60):
            par = np.array([rng.uniform(-400, 400), rng.uniform(-400, 400), rng.uniform(60, 440),
                            rng.uniform(-10, 10), rng.uniform(-0.6, 0.6)])
            wid = rng.integers(0, ch.n_wires, 12)
            d = rng.uniform(0, 1.5, 12)
            r = o.residual(wires, o.hits_of(wid, d), p, par[None], par[None])[0]
            for i in range(12):
                for s, sign in ((0, +1.0), (1, -1.0)):
                    f, Q, e = pm.residual_point(par, _wire_tuple(ch, wid[i]), sign * d[i], x_ref=xr, y_ref=yr, z_ref=z_ref)
                    flo, fhi, scale, decided = r[i, s]
                    if decided:
                        continue
                    if abs(e) > 3.9:           # outside the trig fast range: enclosure is [-1,1] based
                        continue
                    assert flo - 1e-9 * scale <= f <= fhi + 1e-9 * scale, (par, wid[i], s, f, flo, fhi)
                    assert fhi - flo <= 1e-8 * scale


def _sample_box(rng, lo, hi, n):
    pts = rng.uniform(lo, hi, size=(n, 5))
    corners = np.array([[hi[d] if (c >> d) & 1 else lo[d] for d in range(5)] for c in range(32)])
    return np.vstack([corners, pts])


@pytest.mark.parametrize("n", [4, 6])
def test_p5_sampled_range_inside_enclosure(n):
    rng = np.random.default_rng(n)
    ch = g.chamber_c0()
    ev = g.make_event(ch, 0)
    wires = o.wires_of(ch)
    hits = o.hits_of(ev.wire, ev.drift)
    tol = g.TOL
    p = o.make_params(tol)
    n_cells = n ** 5
    cells = rng.choice(n_cells, 40, replace=False)
    blo, bhi = o.cell_boxes(g.BOX_LO, g.BOX_HI, [n] * 5, cells)
    r = o.residual(wires, hits, p, blo, bhi)
    ratios = []
    for ci in range(len(cells)):
        pts = _sample_box(rng, blo[ci], bhi[ci], 1000)
        for h in range(ev.n_hits):
            w = _wire_tuple(ch, ev.wire[h])
            for s, sign in ((0, +1.0), (1, -1.0)):
                flo, fhi, scale, decided = r[ci, h, s]
                if decided:
                    continue
                fs = []
                for dd in (max(ev.drift[h] - tol, 0.0), ev.drift[h] + tol):
                    f, Q, e = pm.residual_point(pts.T, w, sign * dd)
                    fs.append(f[np.abs(e) < 3.9])
                fs = np.concatenate(fs)
                assert fs.min() >= flo - 1e-9 * scale and fs.max() <= fhi + 1e-9 * scale, (cells[ci], h, s)
                if (fs.min() < 0 < fs.max()):
                    assert flo <= 0 <= fhi                          # a sampled sign change must vote
                ratios.append((fhi - flo) / (fs.max() - fs.min()))
    # coarse 4^5 / 6^5 cells are 225 x 225 cm: the dependency problem inflates, but stays bounded
    assert np.median(ratios) < 50


def test_p5_width_ratio_tends_to_one_on_small_boxes():
    rng = np.random.default_rng(2)
    ch = g.chamber_c1()
    ev = g.make_event(ch, 2, smear=0.0)
    wires = o.wires_of(ch)
    hits = o.hits_of(ev.wire, ev.drift)
    tol = g.TOL
    p = o.make_params(tol)
    par = np.array(ev.track.params)
    half = (np.array(g.BOX_HI) - np.array(g.BOX_LO)) / 4096 / 2
    lo, hi = par - half, par + half
    r = o.residual(wires, hits, p, lo[None], hi[None])[0]
    pts = _sample_box(rng, lo, hi, 4000)
    ratios = []
    for h in range(ev.n_hits):
        w = _wire_tuple(ch, ev.wire[h])
        sg, sign = (0, 1.0) if ev.d_true[h] > 0 else (1, -1.0)
        flo, fhi, scale, decided = r[h, sg]
        fs = np.concatenate([pm.residual_point(pts.T, w, sign * dd)[0] for dd in (max(ev.drift[h] - tol, 0), ev.drift[h] + tol)])
        assert fs.min() >= flo and fs.max() <= fhi
        ratios.append((fhi - flo) / (fs.max() - fs.min()))
    assert 1.0 <= min(ratios) and max(ratios) < 1.35, ratios


def test_p6_inclusion_isotonic():
    rng = np.random.default_rng(5)
    ch = g.chamber_c1()
    ev = g.make_event(ch, 3, n_noise=5)
    wires = o.wires_of(ch)
    hits = o.hits_of(ev.wire, ev.drift)
    p = o.make_params(g.TOL)
    lo0, hi0 = np.array(g.BOX_LO), np.array(g.BOX_HI)
    for _ in range(150):
        scale = 2.0 ** -rng.integers(2, 11)
        c = rng.uniform(lo0 + (hi0 - lo0) * scale, hi0 - (hi0 - lo0) * scale)
        plo, phi = c - (hi0 - lo0) * scale / 2, c + (hi0 - lo0) * scale / 2
        f1, f2 = rng.uniform(0, 0.6, 5), rng.uniform(0.4, 1.0, 5)
        clo, chi = plo + (phi - plo) * np.minimum(f1, f2), plo + (phi - plo) * np.maximum(f1, f2)
        rp = o.residual(wires, hits, p, plo[None], phi[None])[0]
        rc = o.residual(wires, hits, p, clo[None], chi[None])[0]
        for h in range(ev.n_hits):
            for s in range(2):
                if rp[h, s, 3]:
                    continue                                  # parent undecidable: votes anyway
                assert not rc[h, s, 3]
                slack = 1e-13 * rp[h, s, 2]                   # libm is not monotone to the last ulp
                assert rc[h, s, 0] >= rp[h, s, 0] - slack and rc[h, s, 1] <= rp[h, s, 1] + slack


def test_fp32_mode_encloses_fp64():
    rng = np.random.default_rng(8)
    ch = g.chamber_c1()
    f32 = lambda a: np.asarray(a, np.float32).astype(np.float64)
    wires = o.wires_of(ch)
    for k in wires.dtype.names:
        wires[k] = f32(wires[k])
    wid = rng.integers(0, ch.n_wires, 20)
    hits = o.hits_of(wid, f32(rng.uniform(0, 1.5, 20)))
    tol = float(np.float32(g.TOL))
    lo0, hi0 = np.array(g.BOX_LO), np.array(g.BOX_HI)
    c = rng.uniform(lo0 * 0.8 + hi0 * 0.2, lo0 * 0.2 + hi0 * 0.8, size=(200, 5))
    w = (hi0 - lo0) * 2.0 ** -rng.integers(3, 9, size=(200, 1))
    blo, bhi = f32(c - w / 2), f32(c + w / 2)
    r64 = o.residual(wires, hits, o.make_params(tol, precision=64), blo, bhi)
    r32 = o.residual(wires, hits, o.make_params(tol, precision=32), blo, bhi)
    ok = (r64[..., 3] == 0) & (r32[..., 3] == 0)
    assert ok.mean() > 0.9
    assert (r32[..., 0][ok] <= r64[..., 0][ok]).all() and (r32[..., 1][ok] >= r64[..., 1][ok]).all()
    # and not absurdly wider: excess below 1e-3 of the residual's own scale (float eps ~ 6e-8 times ~1e2 ops)
    excess = np.maximum(r64[..., 0] - r32[..., 0], r32[..., 1] - r64[..., 1])[ok] / r64[..., 2][ok]
    assert np.median(excess) < 1e-4
