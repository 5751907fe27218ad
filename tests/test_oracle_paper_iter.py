"""Pins of the oracle's pieces of the paper's iteration scheme.

F2a  disk pre-filter (3a,b): every variable occurs once => exact range; compared with the closed form in exact
     rational arithmetic, and with the defining property (a voxel that holds a circle passing within r_disk of the
     origin is kept) by brute force.
F2b  selection of the maximum-vote voxels: special cases whose answer the definition fixes - a single voxel (its
     centre, its half-size), a rectangular block (its centre, its half-extent), a set symmetric about a point, the
     accumulator choice for the sign of lambda, order independence.
F2c  hit finding = condition (4) on one multidimensional interval: equals the (pinned) paper-mode vote of a 1-voxel
     grid hit by hit; an interval around the generated truth finds every genuine hit and rejects far noise.
--   hit mask: masked hits do not vote (vote with mask = vote of the sub-list).
"""
from fractions import Fraction as Fr

import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

LO4, HI4 = np.array(g.BOX_LO[:4]), np.array(g.BOX_HI[:4])


def _disk_exact(lo, hi, r):
    F = Fr
    def sq_minmax(l, h):
        l, h = F(l), F(h)
        mn = F(0) if l <= 0 <= h else min(l * l, h * h)
        return mn, max(l * l, h * h)
    xmn, xmx = sq_minmax(lo[0], hi[0])
    ymn, ymx = sq_minmax(lo[1], hi[1])
    smn, smx = sq_minmax(F(lo[2]) - F(r), F(hi[2]) + F(r))
    return (xmn + ymn - smx) <= 0 <= (xmx + ymx - smn)


def test_f2a_disk_filter_is_the_exact_range_test():
    rng = np.random.default_rng(3)
    dims = (9, 8, 7, 2)
    for trial in range(6):
        lo = np.array([rng.uniform(-450, -50), rng.uniform(-450, -50), rng.uniform(5, 60), -10.0])
        hi = np.array([rng.uniform(50, 450), rng.uniform(50, 450), rng.uniform(100, 450), 10.0])
        r = [10.0, 0.0, 3.5, 25.0, 10.0, 1.0][trial]
        keep = o.disk_filter(lo, hi, dims, r)
        n = int(np.prod(dims))
        blo, bhi = o.cell_boxes4(lo, hi, dims, np.arange(n))
        exact = np.array([_disk_exact(blo[i], bhi[i], r) for i in range(n)])
        # the enclosure is the exact range up to outward rounding: it may only add knife-edge voxels
        assert (keep[exact] == 1).all()
        extra = np.nonzero((keep == 1) & ~exact)[0]
        assert len(extra) <= 2
        assert 0 < keep.sum() < n or r == 25.0
        # defining property by brute force: a circle through a point within r of the origin
        for _ in range(300):
            i = int(rng.integers(n))
            xc, yc = rng.uniform(blo[i, 0], bhi[i, 0]), rng.uniform(blo[i, 1], bhi[i, 1])
            R = rng.uniform(blo[i, 2], bhi[i, 2])
            if abs(np.hypot(xc, yc) - R) <= r * (1 - 1e-12):
                assert keep[i] == 1


def _votes_with(dims, cells, acc, vmax=7, base=3):
    n = int(np.prod(dims))
    v = np.full((2, n), base, np.uint16)
    for c in cells:
        idx = ((c[0] * dims[1] + c[1]) * dims[2] + c[2]) * dims[3] + c[3]
        v[acc, idx] = vmax
    return v


def test_f2b_selection_special_cases():
    dims = (10, 8, 6, 4)
    lo, hi = np.array([-100.0, -80.0, 60.0, -8.0]), np.array([100.0, 80.0, 120.0, 8.0])
    w = (hi - lo) / np.array(dims)
    P = 200.0
    # one voxel: its centre and half-size
    f = o.select_max_paper(_votes_with(dims, [(3, 5, 2, 1)], 0), lo, hi, dims, P)
    assert f.n_sel == 1 and f.vmax == 7 and f.lambda_sign == 1
    assert np.allclose(list(f.value), lo + (np.array([3, 5, 2, 1]) + 0.5) * w, rtol=0, atol=1e-12)
    assert np.allclose(list(f.error), 0.5 * w, rtol=0, atol=1e-12)
    assert abs(f.lam - np.sqrt((P / f.value[2]) ** 2 - 1)) < 1e-12
    # a rectangular block in the other accumulator: its centre, its half-extent, lambda < 0
    block = [(i, j, k, l) for i in (2, 3, 4) for j in (1, 2) for k in (0, 1, 2, 3) for l in (3,)]
    f = o.select_max_paper(_votes_with(dims, block, 1), lo, hi, dims, P)
    assert f.n_sel == len(block) and f.lambda_sign == -1 and f.lam < 0
    assert np.allclose(list(f.value), lo + np.array([3.5, 2.0, 2.0, 3.5]) * w, rtol=0, atol=1e-12)
    assert np.allclose(list(f.error), 0.5 * np.array([3, 2, 4, 1]) * w, rtol=0, atol=1e-12)
    # a set symmetric about a voxel centre (an L-shape and its mirror image): value = that centre
    sym = [(5, 4, 3, 2), (6, 4, 3, 2), (4, 4, 3, 2), (5, 5, 3, 2), (5, 3, 3, 2), (7, 6, 3, 2), (3, 2, 3, 2)]
    f = o.select_max_paper(_votes_with(dims, sym, 0), lo, hi, dims, P)
    assert np.allclose(list(f.value), lo + (np.array([5, 4, 3, 2]) + 0.5) * w, rtol=0, atol=1e-12)
    assert np.allclose(list(f.error), 0.5 * np.array([5, 5, 1, 1]) * w, rtol=0, atol=1e-12)
    # equal maxima in both accumulators: lambda >= 0 wins; a larger maximum in accumulator 1 wins
    v = _votes_with(dims, [(1, 1, 1, 1)], 0)
    v[1] = _votes_with(dims, [(8, 6, 4, 2)], 1)[1]
    f = o.select_max_paper(v, lo, hi, dims, P)
    assert f.lambda_sign == 1 and np.isclose(f.value[0], lo[0] + 1.5 * w[0])
    v[1, 5] = 9
    f = o.select_max_paper(v, lo, hi, dims, P)
    assert f.lambda_sign == -1 and f.vmax == 9 and f.n_sel == 1
    # R value above P: no lambda
    f = o.select_max_paper(_votes_with(dims, [(3, 5, 5, 1)], 0), lo, hi, dims, 100.0)
    assert f.lam == 0.0


def test_f2c_hit_finding_and_hit_mask():
    ch = g.chamber_c1()
    wires = o.wires_of(ch)
    p = o.make_params(g.TOL)
    for seed in (41, 42, 43, 44):
        ev = g.make_event(ch, seed, n_noise=12)
        hits = o.hits_of(ev.wire, ev.drift)
        xc, yc, R, z0, lam = ev.track.params
        P = R * np.sqrt(1 + lam * lam)
        c = np.array([xc, yc, R, z0])
        sgn = 1 if lam >= 0 else -1
        for hw in (np.array([0.3, 0.3, 0.3, 1.0]), np.array([5.0, 5.0, 3.0, 4.0])):
            fl = o.find_hits_paper(wires, hits, p, P, sgn, c - hw, c + hw)
            # definition: the paper-mode vote of the 1-voxel grid, hit by hit
            for h in range(ev.n_hits):
                v = o.vote_paper(wires, hits[h:h + 1], p, P, c - hw, c + hw, (1, 1, 1, 1))
                assert fl[h] == v[0 if sgn > 0 else 1, 0]
            genuine = ~ev.is_noise & ~ev.clipped
            assert fl[genuine].all()
        # the small interval rejects most noise hits
        fl = o.find_hits_paper(wires, hits, p, P, sgn, c - 0.3, c + 0.3)
        assert fl[ev.is_noise].sum() <= 3
        # hit mask = vote of the sub-list; disk filter only removes voxels
        mask = (np.arange(ev.n_hits) % 3 != 0).astype(np.uint8)
        dims = (5, 4, 6, 3)
        vm = o.vote_paper(wires, hits, p, P, LO4, HI4, dims, hit_mask=mask)
        vs = o.vote_paper(wires, hits[mask == 1], p, P, LO4, HI4, dims)
        assert (vm == vs).all()
        vd = o.vote_paper(wires, hits, p, P, LO4, HI4, dims, r_disk=10.0)
        vf = o.vote_paper(wires, hits, p, P, LO4, HI4, dims)
        keep = o.disk_filter(LO4, HI4, dims, 10.0)
        assert (vd[:, keep == 1] == vf[:, keep == 1]).all() and (vd[:, keep == 0] == 0).all()


# ---- paper-shaped workload (8(f) f4), full-turn branch (M6) and the chain (F2e) ----------------------------------------
def test_paper_shaped_generator_against_brute_force():
    """every hit of make_event_paper is a stationary point of the wire-helix distance with DCA <= 0.8 cm, and a dense
    scan of the arc (independent of the generator's candidate search) finds no wire it missed and no closer approach."""
    ch = g.chamber_paper()
    assert ch.n_wires == 5000 and abs(ch.radius[0] - 49.6) < 1e-12 and abs(ch.radius[-1] - 83.7) < 1e-9
    counts = []
    for seed in (0, 1, 2, 3):
        ev = g.make_event_paper(ch, seed)
        trk = ev.track
        assert abs(trk.R * np.sqrt(1 + trk.lam ** 2) - g.PAPER_P) < 1e-12 and trk.z0 == 0.0
        assert 0.45 <= abs(trk.lam) <= 0.85
        counts.append(ev.n_hits)
        assert (ev.drift <= g.PAPER_DRIFT_MAX).all() and (np.abs(ev.z_wire) <= g.PAPER_HALF_LEN).all()
        assert len(set(ev.wire.tolist())) == ev.n_hits
        # dense scan, 0.02 cm steps
        s_end = min(2 * np.pi * trk.R, g.PAPER_HALF_LEN / abs(trk.lam))
        s = np.arange(0.0, s_end, 0.02)
        th = s / trk.R + trk.phi
        hx, hy, hz = trk.xc + trk.R * np.sin(th), trk.yc - trk.R * np.cos(th), trk.lam * s
        T = ch.tan_tau
        wx, wy = ch.sin_phi_s * T, -ch.cos_phi_s * T
        wn = np.sqrt(wx * wx + wy * wy + 1)
        dmin = np.full(ch.n_wires, np.inf)
        for i0 in range(0, len(s), 500):
            sl = slice(i0, i0 + 500)
            qx, qy = hx[None, sl] - ch.x0[:, None], hy[None, sl] - ch.y0[:, None]
            qz = np.broadcast_to(hz[None, sl], qx.shape)
            a = (qx * wx[:, None] + qy * wy[:, None] + qz) / wn[:, None]
            dmin = np.minimum(dmin, np.sqrt(np.maximum(qx * qx + qy * qy + qz * qz - a * a, 0)).min(axis=1))
        hit = np.zeros(ch.n_wires, bool)
        hit[ev.wire] = True
        # the scan (step 0.02 cm along the arc) can only be above the DCA, by at most the half step in quadrature
        assert (dmin[ev.wire] >= ev.drift - 1e-9).all()
        assert (dmin[ev.wire] <= np.sqrt(ev.drift ** 2 + 0.011 ** 2)).all()
        missed = np.nonzero(~hit & (dmin < g.PAPER_DRIFT_MAX - 5e-3))[0]
        # a wire can be missed only if its closest approach lies beyond the end plate (|z on the wire| > half length)
        assert len(missed) <= 2, (seed, missed, dmin[missed])
    assert 15 <= min(counts) and max(counts) <= 65


def test_m6_full_turn_branch_truth_voxel():
    """tracks of more than half a turn (paper-shaped): with the turning angle in [0, 2 pi) (flags bit 3) the truth voxel
    (+-0.5 mm) receives every hit, tol = 0; with the principal value it loses the hits of the returning arc."""
    ch = g.chamber_paper()
    wires = o.wires_of(ch)
    got = {0: 0, 8: 0}
    tot = 0
    for seed in range(8):
        ev = g.make_event_paper(ch, seed)
        xc, yc, R, z0, lam = ev.track.params
        c, hw = np.array([xc, yc, R, z0]), np.array([0.05, 0.05, 0.05, 0.5])
        hits = o.hits_of(ev.wire, ev.drift)
        tot += ev.n_hits
        assert (ev.s_perp / R).max() > np.pi                     # the workload does reach beyond half a turn
        for flags in (0, 8):
            v = o.vote_paper(wires, hits, o.make_params(0.0, flags=flags), g.PAPER_P, c - hw, c + hw, (1, 1, 1, 1))
            got[flags] += int(v[0 if lam >= 0 else 1, 0])
    assert got[8] == tot and got[0] < 0.8 * tot


def test_f2e_chain_is_the_composition_of_its_pinned_pieces():
    """orc_track_paper = vote (masked, disk filter) -> select (per sign) -> find hits -> next pass, recomputed here from the
    individually pinned calls on a small schedule; final sign = larger last maximum."""
    ch = g.chamber_paper()
    wires = o.wires_of(ch)
    p = o.make_params(0.01, flags=8)
    ev = g.make_event_paper(ch, 5, n_noise=4)
    hits = o.hits_of(ev.wire, ev.drift)
    lo, hi = np.array(g.PAPER_BOX_LO), np.array(g.PAPER_BOX_HI)
    spec = [("grid", lo, hi, (12, 12, 8, 6)), ("window", (8.0, 8.0, 3.0, 30.0), (10, 10, 8, 6))]
    fits, sign = o.track_paper(wires, hits, p, g.PAPER_P, 10.0, 5.0, o.make_passes(spec))
    for s, which in ((0, +1), (1, -1)):
        v = o.vote_paper(wires, hits, p, g.PAPER_P, lo, hi, spec[0][3], r_disk=10.0)
        f0 = o.select_max_paper(v, lo, hi, spec[0][3], g.PAPER_P, which)
        assert list(f0.value) == list(fits[0, s]["value"]) and f0.vmax == fits[0, s]["vmax"] and f0.n_sel == fits[0, s]["n_sel"]
        val, err = np.array(f0.value), np.array(f0.error)
        mask = o.find_hits_paper(wires, hits, p, g.PAPER_P, which, val - 5.0 * err, val + 5.0 * err)
        half = np.array(spec[1][1])
        v1 = o.vote_paper(wires, hits, p, g.PAPER_P, val - half, val + half, spec[1][2], hit_mask=mask, r_disk=10.0)
        f1 = o.select_max_paper(v1, val - half, val + half, spec[1][2], g.PAPER_P, which)
        assert list(f1.value) == list(fits[1, s]["value"]) and list(f1.error) == list(fits[1, s]["error"])
        assert f1.vmax == fits[1, s]["vmax"] and f1.lambda_sign == which
    assert sign == (-1 if fits[1, 1]["vmax"] > fits[1, 0]["vmax"] else 1)


# ---- F2d': the reference-point update of L98 ------------------------------------------------------------------------

def _fit(xc, yc, R):
    f = np.zeros(1, o.FIT_DT)
    f[0]["value"] = (xc, yc, R, 0.0)
    return f[0]


def test_f2d_move_ref_special_cases():
    """The new reference point is the z_ref-plane point of the wire of the SELECTED hit that lies closest to the recovered
    circle: cases the definition fixes - a circle drawn through one wire point picks that wire; a masked hit is never
    picked; of two equal hits the first wins; no selected hit leaves the point where it was; the point is on the wire
    line at z = z_ref (independent parametrisation of the wire: (x0, y0, 0) + z (sin phi_s tan tau, -cos phi_s tan tau, 1))."""
    ch = g.chamber_paper()
    wires = o.wires_of(ch)
    rng = np.random.default_rng(8)
    for z_ref in (0.0, 12.5, -30.0):
        p = o.make_params(0.0, x_ref=0.3, y_ref=-0.2, z_ref=z_ref)
        wid = rng.choice(ch.n_wires, size=12, replace=False).astype(np.int32)
        hits = o.hits_of(wid, np.full(12, 0.3))
        T = ch.tan_tau[wid]
        px, py = ch.x0[wid] + z_ref * ch.sin_phi_s[wid] * T, ch.y0[wid] - z_ref * ch.cos_phi_s[wid] * T
        for k in (0, 5, 11):
            c = np.array([px[k] + 21.0, py[k] - 17.0])                      # a circle through wire point k
            R = float(np.hypot(px[k] - c[0], py[k] - c[1]))
            others = np.abs(np.hypot(px - c[0], py - c[1]) - R)
            others[k] = np.inf
            assert others.min() > 1e-6
            idx, xy = o.move_ref_paper(wires, hits, None, p, _fit(c[0], c[1], R))
            assert idx == k and np.allclose(xy, (px[k], py[k]), rtol=0, atol=1e-12)
            if z_ref == 0.0:
                assert xy[0] == ch.x0[wid[k]] and xy[1] == ch.y0[wid[k]]     # no arithmetic at all in the plane z = 0
            else:
                assert abs(xy[0] - ch.x0[wid[k]]) + abs(xy[1] - ch.y0[wid[k]]) > 0.5
            # masked out: the runner-up among the selected hits
            mask = np.ones(12, np.uint8)
            mask[k] = 0
            idx2, xy2 = o.move_ref_paper(wires, hits, mask, p, _fit(c[0], c[1], R))
            assert idx2 == int(np.argmin(others)) and np.allclose(xy2, (px[idx2], py[idx2]), atol=1e-12)
        # the same wire twice: the first of the two
        hits2 = o.hits_of(np.array([wid[3], wid[7], wid[3]], np.int32), np.full(3, 0.1))
        idx, _ = o.move_ref_paper(wires, hits2, None, p, _fit(px[3] + 10.0, py[3], 10.0))
        assert idx == 0
        # nothing selected: the point stays
        idx, xy = o.move_ref_paper(wires, hits, np.zeros(12, np.uint8), p, _fit(0.0, 0.0, 30.0))
        assert idx == -1 and tuple(xy) == (0.3, -0.2)


def test_f2d_truth_voxel_keeps_every_hit_for_any_reference_point_and_emission_point():
    """What makes the update legitimate: the residual does not care where the reference point
    is, as long as z0 is read as "z where the helix is closest to it".  Tracks emitted at the origin, at (5, 0) cm and at
    (0, 5) cm; reference point (0, 0), then the point orc_move_ref_paper picks for the generated circle: the +-0.5 mm
    voxel around (xc, yc, R, z0 of that reference point) receives every noise-free hit (tol = 0) in the accumulator of
    the true sign of lambda - and with z0 NOT re-expressed for the new point it loses hits."""
    ch = g.chamber_paper()
    wires = o.wires_of(ch)
    hw = np.array([0.05, 0.05, 0.05, 0.5])
    lost = tot = 0
    for vertex in ((0.0, 0.0), (5.0, 0.0), (0.0, 5.0)):
        for seed in range(4):
            ev = g.make_event_paper(ch, 40 + seed, vertex=vertex)
            t = ev.track
            hits = o.hits_of(ev.wire, ev.drift)
            good = 0 if t.lam >= 0 else 1
            p0 = o.make_params(0.0, flags=8)
            idx, xy = o.move_ref_paper(wires, hits, None, p0, _fit(t.xc, t.yc, t.R))
            assert idx >= 0
            refs = [(0.0, 0.0), (float(xy[0]), float(xy[1])), (-3.0, 2.0)]
            for xr, yr in refs:
                p = o.make_params(0.0, x_ref=xr, y_ref=yr, flags=8)
                c = np.array([t.xc, t.yc, t.R, t.z0_at(xr, yr, unwrap=True)])
                v = o.vote_paper(wires, hits, p, g.PAPER_P, c - hw, c + hw, (1, 1, 1, 1))
                assert v[good, 0] == ev.n_hits, (vertex, seed, (xr, yr), v[:, 0], ev.n_hits)
            # the old z0 with the new reference point is a different helix
            xr, yr = refs[1]
            p = o.make_params(0.0, x_ref=xr, y_ref=yr, flags=8)
            c = np.array([t.xc, t.yc, t.R, t.z0_at(0.0, 0.0, unwrap=True)])
            v = o.vote_paper(wires, hits, p, g.PAPER_P, c - hw, c + hw, (1, 1, 1, 1))
            lost += ev.n_hits - int(v[good, 0])
            tot += ev.n_hits
    assert lost > 0.5 * tot


def test_f2d_transport_of_z0_between_reference_points():
    """z0 re-expressed for a new reference point (orc_transport_z0) against the generator's own helix: the z of the
    generated track where it is closest to the new point (eventgen.Track.z0_at: eq. (1d)'s phi0 by atan2 of the point
    itself, a different route from the oracle's cross/dot form).  Both angle conventions, emission at and off the axis."""
    ch = g.chamber_paper()
    rng = np.random.default_rng(12)
    for vertex in ((0.0, 0.0), (5.0, 0.0), (0.0, 5.0)):
        for seed in range(6):
            ev = g.make_event_paper(ch, 60 + seed, vertex=vertex)
            t = ev.track
            # reference points on the travelled arc (wire points of hits) for the unwrapped convention ...
            pts = [(float(ch.x0[w]), float(ch.y0[w])) for w in ev.wire[:: max(1, ev.n_hits // 6)]]
            for unwrap, flags in ((True, 8), (False, 0)):
                p = o.make_params(0.0, flags=flags)
                a = pts[0]
                for b_ in pts[1:] + [(0.0, 0.0)]:
                    if not unwrap:
                        # ... the principal-value convention needs the two points within half a turn of each other
                        b_ = (a[0] + rng.uniform(-3, 3), a[1] + rng.uniform(-3, 3))
                    f = _fit(t.xc, t.yc, t.R)
                    f["value"][3] = t.z0_at(a[0], a[1], unwrap=unwrap)
                    f["lam"], f["x_ref"], f["y_ref"] = t.lam, a[0], a[1]
                    got = o.transport_z0(p, f, b_[0], b_[1])
                    want = t.z0_at(b_[0], b_[1], unwrap=unwrap)
                    if not unwrap:
                        # same branch as the start point: compare modulo one turn of z
                        turn = 2.0 * np.pi * t.R * t.lam
                        want = want + turn * round((got - want) / turn)
                    assert abs(got - want) < 1e-9, (vertex, seed, unwrap, a, b_, got, want)


def _helix_point(xc, yc, R, phi, z_e, lam, theta, r=None):
    """Eq. (1a-c) L43-47 written out with the turning angle theta = rho s counted from the emission point (direction phi):
    the helix point, or - r given - the point at distance r from the axis of the helix on the same radius, whose closest
    point of the helix (in the transverse plane) is that helix point."""
    rr = R if r is None else r
    return xc + rr * np.sin(phi + theta), yc - rr * np.cos(phi + theta), z_e + lam * R * theta


@pytest.mark.parametrize("vertex", [(0.0, 0.0), (5.0, 0.0), (0.0, 5.0)])
def test_f2d_z0_against_the_helix_written_out(vertex):
    """Independent of eventgen.Track.z0_at and of the oracle: for a reference point on the radius through the helix point
    of turning angle theta, "z where the helix is closest to the reference point" (eq. (1d)) is z_e + lambda R theta
    by eq. (1c).  Checked three ways for both lambda signs, with theta inside the margin below the emission
    point (-0.3 < theta < 0), near a full turn, and for emission at the origin, (5, 0) and (0, 5) cm (L123):
      (i)   Track.z0_at (the generator's statement of the truth the tests compare fits with),
      (ii)  a brute-force scan of the helix for the point closest to the reference point,
      (iii) orc_transport_z0 (reading F2d'): the difference between two reference points is lambda R (theta_b - theta_a)."""
    rng = np.random.default_rng(int(10 * vertex[0] + vertex[1]) + 3)
    p8 = o.make_params(0.0, flags=8)
    for trial in range(12):
        R = rng.uniform(30.0, 38.0)
        phi = rng.uniform(-np.pi, np.pi)
        lam = rng.uniform(0.2, 1.2) * (1 if trial % 2 else -1)
        z_e = rng.uniform(-20.0, 20.0)
        t = g.Track(R, phi, z_e, lam, vertex[0], vertex[1])
        xc, yc = t.xc, t.yc
        # the angle of the emission point in the convention of the unwrapped mode (from the circle point closest to the axis)
        th_v = np.arctan2(np.sin(phi - np.arctan2(-xc, yc)), np.cos(phi - np.arctan2(-xc, yc)))
        lo_th, hi_th = -0.3 - th_v, 2.0 * np.pi - 0.3 - th_v        # turning angles the convention can express
        thetas = np.concatenate([[lo_th + 1e-3, lo_th + 0.15, -1e-3, 1e-3, hi_th - 1e-3, hi_th - 0.2], rng.uniform(0.0, 5.5, 6)])
        prev = None
        for theta in thetas:
            r = R * rng.uniform(0.6, 1.5)                          # off the circle, on the same radius
            px, py, z_want = _helix_point(xc, yc, R, phi, z_e, lam, theta, r)
            # (i)
            assert abs(t.z0_at(px, py, unwrap=True) - z_want) < 1e-9, (vertex, trial, theta)
            # (ii) brute force over the expressible range of turning angles
            scan = np.linspace(lo_th, hi_th, 400001)
            hx, hy, hz = _helix_point(xc, yc, R, phi, z_e, lam, scan)
            k = int(np.argmin((hx - px) ** 2 + (hy - py) ** 2))
            assert abs(hz[k] - z_want) <= abs(lam) * R * (scan[1] - scan[0]) + 1e-9
            # (iii)
            if prev is not None:
                f = _fit(xc, yc, R)
                f["value"][3], f["lam"], f["x_ref"], f["y_ref"] = prev[2], lam, prev[0], prev[1]
                got = o.transport_z0(p8, f, px, py)
                assert abs(got - z_want) < 1e-9, (vertex, trial, theta, got, z_want)
                assert abs((got - prev[2]) - lam * R * (theta - prev[3])) < 1e-9
            prev = (px, py, z_want, theta)
        # the principal-value convention (flags 0): two reference points less than half a turn apart
        p0 = o.make_params(0.0, flags=0)
        for theta_a, theta_b in ((0.2, 1.9), (2.5, 0.4), (-0.2, 0.3), (3.0, 5.9)):
            ax, ay, za = _helix_point(xc, yc, R, phi, z_e, lam, theta_a, 1.2 * R)
            bx, by, zb = _helix_point(xc, yc, R, phi, z_e, lam, theta_b, 0.8 * R)
            f = _fit(xc, yc, R)
            f["value"][3], f["lam"], f["x_ref"], f["y_ref"] = za, lam, ax, ay
            assert abs(o.transport_z0(p0, f, bx, by) - zb) < 1e-9
