"""Pins of the oracle's PAPER-MODE vote (readings M1-M5 of DESIGN.md).

MP1  the mid-voxel number d_Ax (steps S2-S8 at a point) equals the independent numpy / mpmath point
     model written from Appendix A (tests/pointmodel.py): every term of (A.5b), (A.8).
MP2  identity at the generated truth: the voxel centred on the true helix, momentum fixed to its true
     value, tol = 0, receives every noise-free hit in the accumulator of the true lambda sign - fixes
     lambda(P, R) of M2, the accumulator order and the drift-sign handling.
MP3  axial limit T = 0: d_Ax = d_St (L33-35: "the drift distance ... is the radius of a circle").
MP4  exactness of condition (4): with d_Ax a number every interval variable occurs once, so the enclosure
     is the exact range of (x_Ax - xc)^2 + (y_Ax - yc)^2 - (R + d_Ax)^2 over the voxel: compared with the
     closed form in exact rational arithmetic (nearest point / farthest corner of the rectangle).
MP5  tolerance hull (M4) = union of the two literal evaluations at d - tol and d + tol.
MP6  voxels whose mid radius exceeds P (no lambda) get no vote; index order (z0 fastest); the vote is the
     count over hits of "either drift sign contains 0" of the per-(voxel, hit, sign) enclosures.
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

import pointmodel as pm


def _wire_tuple(ch, wid):
    return (ch.x0[wid], ch.y0[wid], ch.sin_phi_s[wid], ch.cos_phi_s[wid], ch.tan_tau[wid])


def _pm_dax(par, wire, d_signed, mp=None, z_ref=0.0, x_ref=0.0, y_ref=0.0):
    xc, yc, R, z0, lam = par
    x0, y0, sphi, cphi, T = wire
    xA, yA, Q, cA, sA, dphi = pm.axial_quantities(xc, yc, x0, y0, sphi, cphi, T, x_ref, y_ref, z_ref, mp)
    e = pm.phi_series(2, xc, yc, R, z0, lam, d_signed, Q, cA, sA, dphi, T, z_ref, mp)
    f, dAx, u = pm.residual_given_e(e, xc, yc, R, z0, lam, d_signed, Q, cA, sA, dphi, T, z_ref, mp)
    return float(dAx), float(Q - f)


def test_mp1_point_dax_equals_point_model():
    import mpmath as mp
    mp.mp.dps = 40
    rng = np.random.default_rng(11)
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    for z_ref, xr, yr in ((0.0, 0.0, 0.0), (1.5, 2.0, -1.0)):
        p = o.make_params(0.0, xr, yr, z_ref)
        for i in range(80):
            par = np.array([rng.uniform(-400, 400), rng.uniform(-400, 400), rng.uniform(60, 440),
                            rng.uniform(-10, 10), rng.uniform(-0.6, 0.6)])
            wid = int(rng.integers(ch.n_wires))
            if np.hypot(ch.x0[wid] - par[0], ch.y0[wid] - par[1]) < 5.0:
                continue
            d = rng.uniform(0.0, 1.5) * rng.choice([-1.0, 1.0])
            ok, rad, dax = o.dax_point(wires[wid], p, par, d)
            dax_np, rad_np = _pm_dax(par, _wire_tuple(ch, wid), d, None, z_ref, xr, yr)
            assert ok
            assert abs(rad - rad_np) <= 1e-11 * abs(rad_np)
            assert abs(dax - dax_np) <= 1e-9          # sqrt(rad) - R cancels ~3 digits
            if i < 10:
                mpar = [mp.mpf(float(x)) for x in par]
                mw = [mp.mpf(float(x)) for x in _wire_tuple(ch, wid)]
                dax_mp, rad_mp = _pm_dax(mpar, mw, mp.mpf(d), mp, mp.mpf(z_ref), mp.mpf(xr), mp.mpf(yr))
                assert abs(rad - rad_mp) <= 1e-11 * abs(rad_mp)
                assert abs(dax - dax_mp) <= 1e-9


@pytest.mark.parametrize("chamber", [g.chamber_c0, g.chamber_c1, g.chamber_c4])
def test_mp2_truth_voxel_gets_every_hit_in_the_right_accumulator(chamber):
    ch = chamber()
    wires = o.wires_of(ch)
    p = o.make_params(0.0)
    n_pos = n_neg = 0
    for seed in range(20):
        ev = g.make_event(ch, 700 + seed, smear=0.0)
        xc, yc, R, z0, lam = ev.track.params
        P = R * np.sqrt(1.0 + lam * lam)
        hw = np.array([0.01, 0.01, 0.01, 0.05])
        c = np.array([xc, yc, R, z0])
        keep = ~ev.clipped
        hits = o.hits_of(ev.wire[keep], np.abs(ev.d_true[keep]))
        v = o.vote_paper(wires, hits, p, P, c - hw, c + hw, (1, 1, 1, 1))
        good = 0 if lam >= 0 else 1
        assert v[good, 0] == keep.sum(), (seed, v[:, 0], keep.sum())
        if abs(lam) > 0.1:
            assert v[1 - good, 0] < keep.sum()        # the wrong lambda sign misses the stereo layers' z
            n_pos += lam > 0
            n_neg += lam < 0
        # per-sign detail: the true drift sign contains 0, the wrong one does not unless |d| is tiny
        r = o.residual_paper(wires, hits, p, P, c - hw, c + hw)[0]
        for i, dt in enumerate(ev.d_true[keep]):
            ds = 0 if dt > 0 else 1
            flo, fhi, scale, has = r[i, good, ds]
            assert has and flo <= 0.0 <= fhi
            if abs(dt) > 0.05:
                wlo, whi, _, whas = r[i, good, 1 - ds]
                assert (not whas) or wlo > 0 or whi < 0
    assert n_pos > 0 and n_neg > 0


def test_mp3_axial_limit_dax_is_the_drift_distance():
    ch = g.make_chamber(6, 20.0, 5.0, 32, 0.0)
    wires = o.wires_of(ch)
    p = o.make_params(0.0)
    rng = np.random.default_rng(5)
    for _ in range(200):
        par = np.array([rng.uniform(-300, 300), rng.uniform(-300, 300), rng.uniform(60, 440),
                        rng.uniform(-10, 10), rng.uniform(-0.6, 0.6)])
        wid = int(rng.integers(ch.n_wires))
        d = rng.uniform(0.0, 1.5) * rng.choice([-1.0, 1.0])
        ok, rad, dax = o.dax_point(wires[wid], p, par, d)
        assert ok
        assert abs(dax - d) <= 4 * np.spacing(par[2] + abs(d))
        assert abs(rad - (par[2] + d) ** 2) <= 4 * np.spacing(rad)


def _exact_range(xA, yA, lo, hi, dax0, dax1):
    """exact min / max of (xA-xc)^2 + (yA-yc)^2 - (R + dAx)^2 over the voxel and dAx in [dax0, dax1] (R + dAx > 0)."""
    F = Fr
    def dist2_minmax(a, l, h):
        a, l, h = F(a), F(l), F(h)
        near = min(max(a, l), h)
        far = l if abs(a - l) >= abs(a - h) else h
        return (a - near) ** 2, (a - far) ** 2
    xmin, xmax = dist2_minmax(xA, lo[0], hi[0])
    ymin, ymax = dist2_minmax(yA, lo[1], hi[1])
    smin = (F(lo[2]) + F(dax0)) ** 2
    smax = (F(hi[2]) + F(dax1)) ** 2
    assert F(lo[2]) + F(dax0) > 0
    return xmin + ymin - smax, xmax + ymax - smin


def test_mp4_condition_4_enclosure_is_the_exact_range():
    rng = np.random.default_rng(21)
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    p = o.make_params(0.0)
    checked = 0
    for _ in range(150):
        c = np.array([rng.uniform(-400, 400), rng.uniform(-400, 400), rng.uniform(70, 430), rng.uniform(-9, 9)])
        hw = np.array([rng.uniform(0.01, 30), rng.uniform(0.01, 30), rng.uniform(0.01, 10), rng.uniform(0.01, 1)])
        lo, hi = c - hw, c + hw
        wid = int(rng.integers(ch.n_wires))
        d = rng.uniform(0.0, 1.5)
        lam_true = rng.uniform(0.05, 0.6)
        mid = 0.5 * (lo + hi)
        P = mid[2] * np.sqrt(1 + lam_true ** 2)
        hits = o.hits_of([wid], [d])
        r = o.residual_paper(wires, hits, p, P, lo, hi)[0, 0]
        q = P / mid[2]
        lam = np.sqrt(q * q - 1.0)                       # M2, same operations
        for ls, lsign in enumerate((+1.0, -1.0)):
            for ds, dsign in enumerate((+1.0, -1.0)):
                ok, rad, dax = o.dax_point(wires[wid], p, [mid[0], mid[1], mid[2], mid[3], lsign * lam], dsign * d)
                flo, fhi, scale, has = r[ls, ds]
                assert bool(has) == ok
                if not ok:
                    continue
                emin, emax = _exact_range(ch.x0[wid], ch.y0[wid], lo, hi, dax, dax)
                assert Fr(flo) <= emin and emax <= Fr(fhi)
                assert float(emin - Fr(flo)) <= 8 * np.spacing(scale)
                assert float(Fr(fhi) - emax) <= 8 * np.spacing(scale)
                checked += 1
    assert checked > 400


def test_mp5_tolerance_hull_is_the_union_of_the_two_literal_evaluations():
    rng = np.random.default_rng(31)
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    tol = g.TOL
    for _ in range(60):
        c = np.array([rng.uniform(-400, 400), rng.uniform(-400, 400), rng.uniform(70, 430), rng.uniform(-9, 9)])
        hw = np.array([5.0, 5.0, 2.0, 0.5])
        lo, hi = c - hw, c + hw
        wid = int(rng.integers(ch.n_wires))
        d = rng.uniform(0.1, 1.4)
        P = c[2] * 1.1
        rt = o.residual_paper(wires, o.hits_of([wid], [d]), o.make_params(tol), P, lo, hi)[0, 0]
        # d - tol and d + tol as computed by the oracle (round to nearest)
        ra = o.residual_paper(wires, o.hits_of([wid], [d - tol]), o.make_params(0.0), P, lo, hi)[0, 0]
        rb = o.residual_paper(wires, o.hits_of([wid], [d + tol]), o.make_params(0.0), P, lo, hi)[0, 0]
        for ls in range(2):
            for ds in range(2):
                if not (rt[ls, ds, 3] and ra[ls, ds, 3] and rb[ls, ds, 3]):
                    continue
                assert rt[ls, ds, 0] == min(ra[ls, ds, 0], rb[ls, ds, 0])
                assert rt[ls, ds, 1] == max(ra[ls, ds, 1], rb[ls, ds, 1])


def test_mp6_grid_layout_no_lambda_voxels_and_vote_definition():
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    ev = g.make_event(ch, 1, n_noise=5)
    hits = o.hits_of(ev.wire, ev.drift)
    p = o.make_params(g.TOL)
    xc, yc, R, z0, lam = ev.track.params
    P = R * np.sqrt(1 + lam * lam)
    lo, hi, dims = np.array(g.BOX_LO[:4]), np.array(g.BOX_HI[:4]), (6, 5, 7, 3)
    v = o.vote_paper(wires, hits, p, P, lo, hi, dims)
    n = int(np.prod(dims))
    assert v.shape == (2, n) and v.max() <= ev.n_hits and v.max() > 0
    idx = np.array([0, 17, 100, n - 1, 333])
    vs = o.vote_paper(wires, hits, p, P, lo, hi, dims, cell_idx=idx)
    assert (vs == v[:, idx]).all()
    blo, bhi = o.cell_boxes4(lo, hi, dims, np.arange(n))
    # z0 fastest: consecutive voxels differ in z0 only
    assert blo[1, 3] > blo[0, 3] and (blo[1, :3] == blo[0, :3]).all()
    # R_m > P: no lambda, no vote
    rm = 0.5 * (blo[:, 2] + bhi[:, 2])
    assert (rm > P).any() and (v[:, rm > P] == 0).all()
    # vote = number of hits for which either drift sign contains 0
    r = o.residual_paper(wires, hits, p, P, blo[idx], bhi[idx])
    yes = (r[..., 3] > 0) & ~((r[..., 0] > 0) | (r[..., 1] < 0))          # [box, hit, ls, ds]
    cnt = yes.any(axis=3).sum(axis=1)                                      # [box, ls]
    assert (cnt.T == vs).all()
