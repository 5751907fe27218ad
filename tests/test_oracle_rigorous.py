"""Pins of the oracle's rigorous-Phi mode (PAPER.md L187 eq. (A.6); flags bit 4).

R1  at the generated truth, thin box, tol = 0, true drift sign: 0 is in the enclosure for every noise-free hit (the
    strict guarantee of L80 restored), and the enclosure stays thin; the series mode misses zero for some hits
    (its truncation error is not enclosed, reading G3) - so the two modes really differ.
R2  brute force: at random points of a box the point residual with Phi solved from (A.6) by plain fixed-point
    iteration (numpy, written from Appendix A via tests/pointmodel.py) lies inside the box's enclosure.
R3  the containment invariant with tol = 0 on dense grids from 8^5 to 4096^5: the truth cell keeps every hit.
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

import pointmodel as pm

RIG = 16


def _wire_tuple(ch, wid):
    return (ch.x0[wid], ch.y0[wid], ch.sin_phi_s[wid], ch.cos_phi_s[wid], ch.tan_tau[wid])


def _point_f_exact_phi(par, wire, d_signed):
    """f of (A.5a,b) with Phi from (A.6) solved by fixed-point iteration in plain doubles."""
    xc, yc, R, z0, lam = par
    x0, y0, sphi, cphi, T = wire
    xA, yA, Q, cA, sA, dphi = pm.axial_quantities(xc, yc, x0, y0, sphi, cphi, T)
    RA = np.sqrt(Q)
    e = 0.0
    for _ in range(200):
        sinP = (sA * np.cos(e) + cA * np.sin(e)) / RA
        cosP = (cA * np.cos(e) - sA * np.sin(e)) / RA
        u = np.sqrt(1 + 2 * lam * sinP * T + lam ** 2 * T ** 2 + cosP ** 2 * T ** 2)      # (A.3a)
        dl = d_signed / u
        z = z0 + lam * R * (dphi + e) - dl * cosP * T                                      # (A.4c)
        s_t = -z * sA - lam * dl * cA                                                      # (A.7c)
        c_t = z * cA - lam * dl * sA                                                       # (A.7b)
        e_new = np.arctan2(s_t * T, Q + c_t * T)                                           # (A.6)
        if abs(e_new - e) < 1e-16:
            break
        e = e_new
    f, dAx, u = pm.residual_given_e(e, xc, yc, R, z0, lam, d_signed, Q, cA, sA, dphi, T)
    return float(f), float(Q)


@pytest.mark.parametrize("chamber", [g.chamber_c0, g.chamber_c1, g.chamber_c4])
def test_r1_zero_is_enclosed_at_the_truth_with_no_tolerance(chamber):
    ch = chamber()
    wires = o.wires_of(ch)
    missed_series = 0
    n = 0
    for seed in range(15):
        ev = g.make_event(ch, 800 + seed, smear=0.0)
        par = np.array(ev.track.params)
        keep = ~ev.clipped
        hits = o.hits_of(ev.wire[keep], np.abs(ev.d_true[keep]))
        rr = o.residual(wires, hits, o.make_params(0.0, flags=RIG), par[None], par[None])[0]
        rs = o.residual(wires, hits, o.make_params(0.0), par[None], par[None])[0]
        for i, dt in enumerate(ev.d_true[keep]):
            sg = 0 if dt > 0 else 1
            flo, fhi, scale, decided = rr[i, sg]
            assert not decided, (seed, i)
            # the generator's DCA is solved to 1e-12 cm: allow that much around zero
            assert flo <= 1e-9 * scale and fhi >= -1e-9 * scale, (seed, i, flo, fhi)
            assert fhi - flo <= 1e-8 * scale
            slo, shi = rs[i, sg][:2]
            missed_series += (slo > 1e-9 * scale) or (shi < -1e-9 * scale)
            n += 1
    assert missed_series > 0.2 * n          # the unenclosed series error is visible at tol = 0


def test_r2_point_residuals_with_solved_phi_lie_inside_the_enclosure():
    rng = np.random.default_rng(17)
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    p = o.make_params(0.0, flags=RIG)
    checked = 0
    for _ in range(40):
        c = np.array([rng.uniform(-300, 300), rng.uniform(-300, 300), rng.uniform(90, 400), rng.uniform(-8, 8),
                      rng.uniform(-0.5, 0.5)])
        hw = np.array([2.0, 2.0, 1.0, 0.3, 0.02]) * rng.uniform(0.05, 1.0)
        lo, hi = c - hw, c + hw
        wid = int(rng.integers(ch.n_wires))
        if np.hypot(ch.x0[wid] - c[0], ch.y0[wid] - c[1]) < 20.0:
            continue
        d = rng.uniform(0.05, 1.4)
        r = o.residual(wires, o.hits_of([wid], [d]), p, lo[None], hi[None])[0, 0]
        for sg, ds in ((0, d), (1, -d)):
            flo, fhi, scale, decided = r[sg]
            if decided:
                continue
            pts = [lo + (hi - lo) * rng.uniform(0, 1, 5) for _ in range(30)]
            pts += [np.where(rng.integers(0, 2, 5) > 0, hi, lo) for _ in range(16)]
            for pt in pts:
                f, Q = _point_f_exact_phi(pt, _wire_tuple(ch, wid), ds)
                assert flo - 1e-9 * scale <= f <= fhi + 1e-9 * scale
                checked += 1
    assert checked > 1500


def test_r3_containment_with_no_tolerance_on_dense_grids():
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    LO, HI = np.array(g.BOX_LO), np.array(g.BOX_HI)
    p = o.make_params(0.0, flags=RIG)
    for seed in range(5):
        ev = g.make_event(ch, 950 + seed, smear=0.0)
        keep = ~ev.clipped
        hits = o.hits_of(ev.wire[keep], np.abs(ev.d_true[keep]))
        for n in (8, 100, 4096):
            dims = (n,) * 5
            tc = g.truth_cell(ev.track.params, LO, HI, dims)
            v = o.vote(wires, hits, p, LO, HI, dims, cell_idx=[tc])
            assert v[0] == keep.sum(), (seed, n, v[0], keep.sum())
