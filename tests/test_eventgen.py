"""Pins for the seeded input generator and for the paper's equations themselves (no oracle here).

P2  worked example (tests/golden/p2_dca_worked_example.txt)
--  independent brute-force minimisation of the helix-wire distance in mpmath
--  (A.3a), (A.4a-c), (A.5a,b), (A.6) hold at the generated closest approach (exact Phi)
P8  series order: error of (A.8) order 1 ~ T^2, order 2 ~ T^3
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2401_04576_b200 import eventgen as g

import pointmodel as pm

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_p2():
    rows = []
    for line in open(os.path.join(GOLD, "p2_dca_worked_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        l, j, d, s = line.split()
        rows.append((int(l), int(j), float(d), float(s)))
    return rows


def test_splitmix64_reference_values():
    # first outputs of splitmix64 seeded with 0 (values of the public reference implementation)
    r = g.SplitMix64(0)
    assert [r.next_u64() for _ in range(3)] == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]
    r = g.SplitMix64(1234567)
    assert [r.next_u64() for _ in range(2)] == [6457827717110365317, 3203168211198807973]


def test_p2_worked_example():
    ch = g.chamber_c0()
    trk = g.Track(200.0, 0.7, 1.25, -0.35)
    assert abs(trk.xc - (-128.84353744753821)) < 1e-12 and abs(trk.yc - 152.96843745689769) < 1e-12
    w, d, s, z = g.track_hits(trk, ch)
    for (l, j, dref, sref), wi, di, si in zip(_read_p2(), w, d, s):
        assert wi == l * 64 + j
        assert abs(di - dref) < 2e-13
        assert abs(si - sref) < 1e-4
    assert abs(z[0] - (-5.8157)) < 1e-4 and abs(z[-1] - (-15.4636)) < 1e-4


def test_dca_against_mpmath_minimisation():
    """The generator's DCA equals a 40-digit minimisation of |M(s) - W(zw)| over (s, zw)."""
    mp.mp.dps = 40
    ch = g.chamber_c1()
    ev = g.make_event(ch, 77, smear=0.0)
    t = ev.track
    for i in (0, 7, 19):
        wid = int(ev.wire[i])
        X0, Y0 = mp.mpf(ch.x0[wid]), mp.mpf(ch.y0[wid])
        sp, cp, T = mp.mpf(ch.sin_phi_s[wid]), mp.mpf(ch.cos_phi_s[wid]), mp.mpf(ch.tan_tau[wid])
        R, phi, z0, lam = map(mp.mpf, (t.R, t.phi, t.z0, t.lam))
        xc, yc = -R * mp.sin(phi), R * mp.cos(phi)

        def grad(s, zw):
            th = s / R + phi
            dx = xc + R * mp.sin(th) - (X0 + zw * sp * T)
            dy = yc - R * mp.cos(th) - (Y0 - zw * cp * T)
            dz = z0 + lam * s - zw
            return (dx * mp.cos(th) + dy * mp.sin(th) + dz * lam, dx * sp * T - dy * cp * T + dz)

        s, zw = mp.findroot(grad, (mp.mpf(ev.s_perp[i]), mp.mpf(ev.z_wire[i])))
        th = s / R + phi
        dist = mp.sqrt((xc + R * mp.sin(th) - (X0 + zw * sp * T)) ** 2 + (yc - R * mp.cos(th) - (Y0 - zw * cp * T)) ** 2
                       + (z0 + lam * s - zw) ** 2)
        assert abs(float(dist) - abs(ev.d_true[i])) < 1e-12
        assert abs(float(s) - ev.s_perp[i]) < 1e-9


def test_nearest_wire_is_global_minimum():
    ch = g.chamber_c4()
    for seed in range(12):
        ev = g.make_event(ch, seed, smear=0.0)
        w_all, _, _, _ = g.track_hits(ev.track, ch, n_cand=ch.wires_per_layer)
        assert (w_all == ev.wire).all()


@pytest.mark.parametrize("chamber", [g.chamber_c0, g.chamber_c1, g.chamber_c4])
@pytest.mark.parametrize("z_ref", [0.0, 3.0])
def test_paper_identities_hold_at_closest_approach(chamber, z_ref):
    """With the exact Phi = rho s + phi0 - phi_s of the closest approach: (A.3a) is |w x t|, and the
    circle equation (A.5a,b) vanishes.  Fixes every sign of (A.3)-(A.7) and the u_d orientation."""
    ch = chamber()
    for seed in range(6):
        ev = g.make_event(ch, 100 + seed, smear=0.0)
        t = ev.track
        xc, yc, R, z0, lam = t.params
        for i in range(ev.n_hits):
            wid = int(ev.wire[i])
            wire = (ch.x0[wid], ch.y0[wid], ch.sin_phi_s[wid], ch.cos_phi_s[wid], ch.tan_tau[wid])
            xA, yA, Q, cA, sA, dphi = pm.axial_quantities(xc, yc, *wire, z_ref=z_ref)
            phi_s = math.atan2(wire[2], wire[3])
            Phi = ev.s_perp[i] / R + t.phi - phi_s
            PhiA = math.atan2(sA, cA)
            e = math.remainder(Phi - PhiA, 2 * math.pi)
            f, dAx, u = pm.residual_given_e(e, xc, yc, R, z0, lam, ev.d_true[i], Q, cA, sA, dphi, wire[4], z_ref=z_ref)
            assert abs(f) <= 1e-9 * Q, (seed, i, f, Q)
            # (A.3a) is the norm of w x t
            th = ev.s_perp[i] / R + t.phi
            w = np.array([wire[2] * wire[4], -wire[3] * wire[4], 1.0])
            tv = np.array([math.cos(th), math.sin(th), lam])
            assert abs(u - np.linalg.norm(np.cross(w, tv))) < 1e-13
            # (A.6): Phi = Phi_Ax + atan2(s^tau T, RAx^2 + c^tau T)
            dl = ev.d_true[i] / u
            zst = z0 + lam * ev.s_perp[i] - z_ref - dl * math.cos(Phi) * wire[4]
            ctau = -lam * dl * sA + zst * cA
            stau = -lam * dl * cA - zst * sA
            assert abs(e - math.atan2(stau * wire[4], Q + ctau * wire[4])) < 1e-12


def test_p8_series_order():
    """Halving tau: the order-1 truncation error of (A.8) falls ~4x, the order-2 error ~8x."""
    errs = {1: [], 2: []}
    taus = [0.1, 0.05, 0.025, 0.0125]
    trk = g.Track(150.0, 1.1, 2.0, 0.45)
    for tau in taus:
        ch = g.make_chamber(8, 20.0, 4.0, 64, tau)
        w, d, s, z = g.track_hits(trk, ch)
        xc, yc, R, z0, lam = trk.params
        for order in (1, 2):
            worst = 0.0
            for wid, di, si in zip(w, d, s):
                wire = (ch.x0[wid], ch.y0[wid], ch.sin_phi_s[wid], ch.cos_phi_s[wid], ch.tan_tau[wid])
                xA, yA, Q, cA, sA, dphi = pm.axial_quantities(xc, yc, *wire)
                e = pm.phi_series(order, xc, yc, R, z0, lam, di, Q, cA, sA, dphi, wire[4])
                Phi = si / R + trk.phi - math.atan2(wire[2], wire[3])
                e_true = math.remainder(Phi - math.atan2(sA, cA), 2 * math.pi)
                worst = max(worst, abs(e - e_true))
            errs[order].append(worst)
    r1 = [errs[1][i] / errs[1][i + 1] for i in range(3)]
    r2 = [errs[2][i] / errs[2][i + 1] for i in range(3)]
    assert all(2.5 < r < 5.5 for r in r1) and r1[-1] > 3.5, (errs[1], r1)
    assert all(5.5 < r < 11.0 for r in r2) and r2[-1] > 7.0, (errs[2], r2)
    assert errs[2][0] < errs[1][0]


def test_config_shapes_and_determinism():
    c0 = g.config(0)
    assert c0.chamber.n_wires == 512 and c0.events[0].n_hits == 8 and c0.grid == (16,) * 5
    c1 = g.config(1)
    assert c1.chamber.n_wires == 2560 and c1.events[0].n_hits == 40 and c1.k == 10
    c3 = g.config(3, n_events=3)
    assert [e.n_hits for e in c3.events] == [30, 30, 30] and c3.levels == 8 and c3.k == 8
    c4 = g.config(4)
    assert c4.chamber.n_wires == 10240 and c4.events[0].n_hits == 60 and c4.n_cells == 64 ** 5
    again = g.config(4).events[0]
    assert (again.wire == c4.events[0].wire).all() and (again.drift == c4.events[0].drift).all()
    ev = c1.events[0]
    assert ((ev.drift >= 0) & (ev.drift <= g.DRIFT_MAX)).all()
    assert ev.is_noise.sum() == 20 and (ev.wire[ev.is_noise] < 2560).all()
    # track distributions
    for seed in range(50):
        t = g.make_track(g.SplitMix64(seed))
        assert 80 <= t.R <= 400 and 0 <= t.phi < 2 * math.pi and abs(t.lam) <= 0.5


def test_cell_edges_and_truth_cell():
    e = g.cell_edges(-450.0, 450.0, 16)
    assert e[0] == -450.0 and e[-1] == 450.0 and np.all(e == -e[::-1])
    trk = g.Track(200.0, 0.7, 1.25, -0.35)
    assert g.truth_cell(trk.params, g.BOX_LO, g.BOX_HI, (4,) * 5) == 408
    assert g.truth_cell(trk.params, g.BOX_LO, g.BOX_HI, (16,) * 5) == 370323
