"""Pins of the oracle's vote, top-K and refinement (steps S1, S9) - no GPU.

P3  containment: the cell holding the generated truth gets the vote of every unclipped noise-free
    genuine hit at every grid size from 8^5 down to range/4096 ("when the
    condition (4) is false the solution is not in the voxel").
P4  axial limit (section 2.1): tan(tau)=0 collapses the residual to the textbook
    circle-tangency test, whose interval range is exact; compared with exact rational arithmetic.
P7  symmetry: rotating wires and the (xc,yc) grid by 90 degrees permutes the accumulator.
P9  DAG anchor: vote histograms of the P2 event (tests/golden/p9_dag_anchor.txt).
--  top-K against numpy lexsort, refinement against its definition (children, order, centre).
"""
import os
from fractions import Fraction as F

import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LO, HI = np.array(g.BOX_LO), np.array(g.BOX_HI)


def _p2_event():
    rows = [l.split() for l in open(os.path.join(GOLD, "p2_dca_worked_example.txt")) if l.strip() and l[0] != "#"]
    wire = np.array([int(r[0]) * 64 + int(r[1]) for r in rows], np.int32)
    drift = np.array([abs(float(r[2])) for r in rows])
    return wire, drift


def _read_p9():
    out = {}
    for line in open(os.path.join(GOLD, "p9_dag_anchor.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, hist, tot, truth, top = [s.strip() for s in line.split("|")]
        out[int(n)] = (np.array(hist.split(), np.int64), int(tot), int(truth),
                       None if top == "-" else np.array(top.split(), np.int64))
    return out


@pytest.mark.parametrize("n", [4, 8, 16])
def test_p9_dag_anchor(n):
    hist_ref, tot_ref, truth_idx, top_ref = _read_p9()[n]
    ch = g.chamber_c0()
    wire, drift = _p2_event()
    votes = o.vote(o.wires_of(ch), o.hits_of(wire, drift), o.make_params(g.TOL), LO, HI, [n] * 5)
    hist = np.bincount(votes, minlength=9)
    # the anchor was evaluated in round-to-nearest: outward rounding may move a handful of
    # knife-edge cells; a DAG/convention error moves hundreds
    assert np.abs(hist - hist_ref).sum() <= max(4, n ** 5 // 50000), (hist, hist_ref)
    assert abs(int(votes.sum()) - tot_ref) <= max(4, n ** 5 // 50000)
    assert votes.sum() >= tot_ref or np.abs(hist - hist_ref).sum() > 0 or votes.sum() == tot_ref
    assert votes[truth_idx] == 8
    if top_ref is not None:
        idx, v = o.topk(votes, 10)
        assert (idx == top_ref).all() and (v == 8).all()


@pytest.mark.parametrize("chamber,tol", [(g.chamber_c0, g.TOL), (g.chamber_c1, g.TOL), (g.chamber_c1, 1e-4),
                                         (g.chamber_c4, 1e-4)])
def test_p3_containment(chamber, tol):
    ch = chamber()
    wires = o.wires_of(ch)
    p = o.make_params(tol)
    for seed in range(6):
        ev = g.make_event(ch, 300 + seed, smear=0.0)
        ok = ~ev.clipped
        hits = o.hits_of(ev.wire, ev.drift)
        for level in range(10):
            n = 8 << level
            cell = g.truth_cell(ev.track.params, LO, HI, (n,) * 5)
            blo, bhi = o.cell_boxes(LO, HI, [n] * 5, [cell])
            assert (blo[0] <= ev.track.params).all() and (ev.track.params <= bhi[0]).all()
            r = o.residual(wires, hits, p, blo, bhi)[0]
            for i in np.nonzero(ok)[0]:
                s = 0 if ev.d_true[i] > 0 else 1
                flo, fhi, scale, decided = r[i, s]
                assert decided or (flo <= 0.0 <= fhi), (seed, level, i, flo, fhi)
            v = o.vote(wires, hits, p, LO, HI, [n] * 5, cell_idx=[cell])
            assert v[0] >= ok.sum()


def _exact_axial_vote(xA, yA, d, tol, blo, bhi):
    """0 in (xA-X)^2 + (yA-Y)^2 - (R + D)^2 for D = +/-[max(d-tol,0), d+tol], exact rationals.
    Every variable occurs once, so the natural interval extension is the exact range.
    Returns (vote, margin) with margin = relative distance of the nearest endpoint pair."""
    X, Y, R = (F(blo[0]), F(bhi[0])), (F(blo[1]), F(bhi[1])), (F(blo[2]), F(bhi[2]))

    def sq_range(a):
        lo, hi = a
        if lo >= 0:
            return lo * lo, hi * hi
        if hi <= 0:
            return hi * hi, lo * lo
        return F(0), max(lo * lo, hi * hi)

    A = (F(xA) - X[1], F(xA) - X[0])
    B = (F(yA) - Y[1], F(yA) - Y[0])
    qa, qb = sq_range(A), sq_range(B)
    Q = (qa[0] + qb[0], qa[1] + qb[1])
    Dp = (max(F(d) - F(tol), F(0)), F(d) + F(tol))
    vote, margin = False, None
    for D in (Dp, (-Dp[1], -Dp[0])):
        rad = sq_range((R[0] + D[0], R[1] + D[1]))
        flo, fhi = Q[0] - rad[1], Q[1] - rad[0]
        vote |= flo <= 0 <= fhi
        m = min(abs(flo), abs(fhi)) / max(Q[1], rad[1])
        margin = m if margin is None else min(margin, m)
    return vote, float(margin)


def test_p4_axial_limit_closed_form():
    rng = np.random.default_rng(4)
    ch = g.make_chamber(8, 20.0, 4.0, 64, 0.0)          # axial chamber: tan(tau) = 0
    assert (ch.tan_tau == 0).all()
    wires = o.wires_of(ch)
    tol = g.TOL
    p = o.make_params(tol)
    wid = rng.integers(0, ch.n_wires, 6)
    d = rng.uniform(0, 1.5, 6)
    d[0] = 0.01                                          # d - tol < 0: the clamp at 0
    hits = o.hits_of(wid, d)
    n_box, n_yes, n_no, n_dec = 1500, 0, 0, 0
    c = rng.uniform(LO, HI, size=(n_box, 5))
    # centre half of the boxes on a circle tangent to a wire circle so that votes are not all "no"
    for i in range(0, n_box, 2):
        h = rng.integers(0, 6)
        ang, Rr = rng.uniform(0, 2 * np.pi), rng.uniform(60, 440)
        rr = Rr + rng.choice([-1, 1]) * d[h]
        c[i, 0], c[i, 1], c[i, 2] = ch.x0[wid[h]] + rr * np.cos(ang), ch.y0[wid[h]] + rr * np.sin(ang), Rr
    w = (HI - LO) * 2.0 ** -rng.integers(4, 16, size=(n_box, 1))
    blo, bhi = c - w / 2, c + w / 2
    blo[:, 2] = np.maximum(blo[:, 2], 10.0)
    blo[:, 4], bhi[:, 4] = np.maximum(blo[:, 4], -0.6), np.minimum(bhi[:, 4], 0.6)
    r = o.residual(wires, hits, p, blo, bhi)
    for i in range(n_box):
        for h in range(6):
            exact, margin = _exact_axial_vote(ch.x0[wid[h]], ch.y0[wid[h]], d[h], tol, blo[i], bhi[i])
            got = any(r[i, h, s, 3] or (r[i, h, s, 0] <= 0 <= r[i, h, s, 1]) for s in range(2))
            if r[i, h, 0, 3]:
                # the xy cell contains the wire point: R_Ax^2 reaches 0 and 1/R_Ax^2 of (A.8b,c) is
                # undefined, so the hit cannot be excluded and votes (reading G15)
                assert F(blo[i, 0]) <= F(ch.x0[wid[h]]) <= F(bhi[i, 0]) and F(blo[i, 1]) <= F(ch.y0[wid[h]]) <= F(bhi[i, 1])
                n_dec += 1
                continue
            if margin > 1e-13:
                assert got == exact, (i, h, margin)
            else:
                assert got or not exact               # knife edge: outward rounding may only add a vote
            n_yes += exact
            n_no += not exact
    assert n_yes > 300 and n_no > 300 and n_dec < 50


def test_p7_rotation_by_90_degrees_permutes_votes():
    n = 8
    ch = g.chamber_c0()
    ev = g.make_event(ch, 0)
    wires = o.wires_of(ch)
    rot = wires.copy()                                   # (x,y) -> (-y,x); phi_s -> phi_s + pi/2
    rot["x0"], rot["y0"] = -wires["y0"], wires["x0"]
    rot["sin_phi_s"], rot["cos_phi_s"] = wires["cos_phi_s"], -wires["sin_phi_s"]
    hits = o.hits_of(ev.wire, ev.drift)
    p = o.make_params(g.TOL)
    v = o.vote(wires, hits, p, LO, HI, [n] * 5).reshape(n, n, n, n, n)
    vr = o.vote(rot, hits, p, LO, HI, [n] * 5).reshape(n, n, n, n, n)
    # cell (ix,iy) of the original = cell (n-1-iy, ix) of the rotated problem
    expect = np.flip(v, axis=1).transpose(1, 0, 2, 3, 4)
    assert (vr == expect).all()
    assert 0 < (v == 8).sum() < v.size


def test_topk_matches_lexsort_and_ties_break_on_index():
    rng = np.random.default_rng(1)
    votes = rng.integers(0, 6, 5000).astype(np.uint16)
    order = np.lexsort((np.arange(len(votes)), -votes.astype(np.int64)))
    for k in (1, 7, 16, 500):
        idx, v = o.topk(votes, k)
        assert (idx == order[:k]).all() and (v == votes[order[:k]]).all()
    idx, v = o.topk(np.zeros(40, np.uint16), 5)
    assert (idx == np.arange(5)).all()
    with pytest.raises(RuntimeError):
        o.topk(votes[:3], 4)


def test_refine_follows_its_definition():
    ch = g.chamber_c1()
    ev = g.make_event(ch, 2, n_noise=6)
    wires, hits, p = o.wires_of(ch), o.hits_of(ev.wire, ev.drift), o.make_params(g.TOL)
    grid0, levels, k = [4] * 5, 4, 5
    boxes, par = o.refine(wires, hits, p, LO, HI, grid0, levels, k)
    assert boxes.shape == (levels, k)
    # level 0 = top-K of the dense start grid
    v0 = o.vote(wires, hits, p, LO, HI, grid0)
    idx, vv = o.topk(v0, k)
    blo, bhi = o.cell_boxes(LO, HI, grid0, idx)
    assert (boxes[0]["lo"] == blo).all() and (boxes[0]["hi"] == bhi).all() and (boxes[0]["votes"] == vv).all()
    for lev in range(1, levels):
        # children of the previous level's boxes, list index rank*32+c, bit (4-dim) of c -> upper half
        clo, chi = [], []
        for r in range(k):
            lo, hi = boxes[lev - 1][r]["lo"], boxes[lev - 1][r]["hi"]
            mid = 0.5 * (lo + hi)
            for c in range(32):
                up = np.array([(c >> (4 - d)) & 1 for d in range(5)], bool)
                clo.append(np.where(up, mid, lo))
                chi.append(np.where(up, hi, mid))
        clo, chi = np.array(clo), np.array(chi)
        cv = o.vote_boxes(wires, hits, p, clo, chi)
        idx, vv = o.topk(cv, k)
        assert (boxes[lev]["lo"] == clo[idx]).all() and (boxes[lev]["hi"] == chi[idx]).all()
        assert (boxes[lev]["votes"] == vv).all()
        assert boxes[lev]["votes"].max() <= boxes[lev - 1]["votes"].max()          # P6
        assert (np.diff(boxes[lev]["votes"].astype(int)) <= 0).all()
    last = boxes[-1][0]
    assert (par[:5] == 0.5 * (last["lo"] + last["hi"])).all() and (par[5:10] == 0.5 * (last["hi"] - last["lo"])).all()
    assert np.allclose(par[5:10], (HI - LO) / 4 / 2 ** (levels - 1) / 2)
    # G19: hull of the kept boxes of the last pass that share the maximum vote count (written out from its definition)
    top = boxes[-1][boxes[-1]["votes"] == boxes[-1]["votes"].max()]
    assert (par[10:15] == top["lo"].min(axis=0)).all() and (par[15:20] == top["hi"].max(axis=0)).all()
    assert (par[10:15] <= last["lo"]).all() and (par[15:20] >= last["hi"]).all()


def test_refine_batch_equals_loop_and_fp32_runs():
    ch = g.chamber_c1()
    evs = [g.make_event(ch, 1000 + e, n_noise=3) for e in range(3)]
    wires, p = o.wires_of(ch), o.make_params(g.TOL)
    hits = o.hits_of(np.concatenate([e.wire for e in evs]), np.concatenate([e.drift for e in evs]))
    off = np.cumsum([0] + [e.n_hits for e in evs]).astype(np.int32)
    boxes, par = o.refine_batch(wires, hits, off, p, LO, HI, [4] * 5, 3, 4)
    for e, ev in enumerate(evs):
        b1, p1 = o.refine(wires, o.hits_of(ev.wire, ev.drift), p, LO, HI, [4] * 5, 3, 4)
        assert (boxes[e]["lo"] == b1["lo"]).all() and (boxes[e]["votes"] == b1["votes"]).all() and (par[e] == p1).all()
    p32 = o.make_params(g.TOL, precision=32)
    v64 = o.vote(wires, o.hits_of(evs[0].wire, evs[0].drift), p, LO, HI, [4] * 5)
    v32 = o.vote(wires, o.hits_of(evs[0].wire, evs[0].drift), p32, LO, HI, [4] * 5)
    # float enclosures are wider: they can only add votes (inputs here are not float-exact, so allow a few)
    assert (v32 >= v64).mean() > 0.999 and (v32 == v64).mean() > 0.9


def test_domain_and_argument_errors():
    ch = g.chamber_c0()
    wires, p = o.wires_of(ch), o.make_params(g.TOL)
    hits = o.hits_of([3], [0.5])
    with pytest.raises(RuntimeError):
        o.vote(wires, o.hits_of([9999], [0.5]), p, LO, HI, [2] * 5)          # unknown wire
    lo = LO.copy()
    lo[2] = 0.0
    with pytest.raises(RuntimeError):
        o.vote(wires, hits, p, lo, HI, [2] * 5)                               # R.lo <= 0
    hi = HI.copy()
    hi[4] = 6.0
    with pytest.raises(RuntimeError):
        o.vote(wires, hits, p, LO, hi, [2] * 5)                               # |lambda| tan(tau) >= 0.5
    assert o.vote(wires, o.hits_of([], []), p, LO, HI, [2] * 5).sum() == 0   # no hits: zero votes
