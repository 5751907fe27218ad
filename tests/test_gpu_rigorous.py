"""-m gpu parity of the rigorous-Phi mode (IA_FLAG_RIGOROUS_PHI) against the oracle's.

Same algorithm on both sides (verification of the fixed point of (A.6) by inflation from the series enclosure, then
S5-S8); they differ only in the padding of sin, cos and atan2, a few ulps per round of the verification.
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import binding as b
from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

from gpu_common import HI, LO, Rig, compare_votes

pytestmark = pytest.mark.gpu
RIG = b.FLAG_RIGOROUS_PHI


@pytest.mark.parametrize("precision", [64, 32])
def test_rigorous_residual_enclosures_match(precision):
    rng = np.random.default_rng(23)
    rig = Rig(g.chamber_c1(), precision=precision, flags=RIG)
    try:
        ev = g.make_event(rig.ch, 6, n_noise=10)
        hd, oh = rig.hits(ev.wire, ev.drift)
        par = np.array(ev.track.params)
        n = 500
        c = np.stack([rng.uniform(LO, HI) for _ in range(n)])
        half = (HI - LO)[None, :] * 2.0 ** -rng.integers(3, 12, (n, 1)).astype(np.float64) / 2
        for i in range(200):
            c[i] = par + rng.uniform(-1, 1, 5) * half[i]
        blo, bhi = c - half, c + half
        blo[:, 2] = np.maximum(blo[:, 2], 20.0)
        blo[:, 4], bhi[:, 4] = np.maximum(blo[:, 4], -0.6), np.minimum(bhi[:, 4], 0.6)
        rg = rig.gpu_residual(hd, len(oh), blo, bhi)
        ro = o.residual(rig.owires, oh, rig.oparams, blo, bhi)
        same_forced = rg[..., 3] == ro[..., 3]
        assert same_forced.mean() > 0.9995                  # "verified in round k" can flip on an ulp
        live = (ro[..., 3] == 0) & same_forced
        tol = (1e-12 if precision == 64 else 5e-4) * ro[..., 2]
        assert (np.abs(rg[..., 0] - ro[..., 0])[live] <= tol[live]).mean() > 0.9995
        assert (np.abs(rg[..., 1] - ro[..., 1])[live] <= tol[live]).mean() > 0.9995
        vg = (rg[..., 3] == 1) | ((rg[..., 0] <= 0) & (rg[..., 1] >= 0))
        vo = (ro[..., 3] == 1) | ((ro[..., 0] <= 0) & (ro[..., 1] >= 0))
        assert (vg == vo).mean() > 0.9995 and vg.any() and not vg.all()
    finally:
        rig.close()


def test_rigorous_dense_vote_refine_and_truth_with_no_tolerance():
    """dense 12^5 vote (every cell, mismatches traced), a 4-level refinement (boxes identical), and the strict
    guarantee: with tol = 0 the cell holding the generated parameters keeps every noise-free hit at every size."""
    rig = Rig(g.chamber_c1(), flags=RIG)
    try:
        ev = g.make_event(rig.ch, 1, n_noise=20)
        hd, oh = rig.hits(ev.wire, ev.drift)
        dims = (12,) * 5
        vg = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
        rig.ctx.synchronize()
        vg = vg.cpu().numpy()
        vo = o.vote(rig.owires, oh, rig.oparams, LO, HI, dims)
        compare_votes(rig, hd, oh, vg, vo, lambda idx: o.cell_boxes(LO, HI, dims, idx))
        # the mode is really on: it differs from the series mode in thousands of cells
        rig.ctx.ia_set_params(g.TOL, flags=0)
        vs = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
        rig.ctx.synchronize()
        assert (vs.cpu().numpy() != vg).sum() > 1000
        rig.ctx.ia_set_params(g.TOL, flags=RIG)
        boxes, par = rig.ctx.ia_refine(hd, ev.n_hits, LO, HI, (8,) * 5, 4, 8)
        rig.ctx.synchronize()
        gb = b.boxes_to_numpy(boxes, (4, 8))
        ob, opar = o.refine(rig.owires, oh, rig.oparams, LO, HI, (8,) * 5, 4, 8)
        assert (gb["lo"] == ob["lo"]).all() and (gb["hi"] == ob["hi"]).all() and (gb["votes"] == ob["votes"]).all()
        assert (par.cpu().numpy() == opar).all()
    finally:
        rig.close()
    rig = Rig(g.chamber_c1(), tol=0.0, flags=RIG)
    try:
        for seed in range(4):
            ev = g.make_event(rig.ch, 960 + seed, smear=0.0)
            keep = ~ev.clipped
            hd, oh = rig.hits(ev.wire[keep], np.abs(ev.d_true[keep]))
            for n in (8, 100, 4096):
                dims = (n,) * 5
                tc = g.truth_cell(ev.track.params, LO, HI, dims)
                blo, bhi = o.cell_boxes(LO, HI, dims, [tc])
                v = rig.ctx.ia_vote_boxes(hd, int(keep.sum()), rig.dev(blo), rig.dev(bhi))
                rig.ctx.synchronize()
                assert int(v.cpu().numpy()[0]) == keep.sum(), (seed, n)
    finally:
        rig.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_sign_specialised_rigorous_kernel_agrees_with_the_general_one(precision):
    """IA_FLAG_RIGOROUS_PHI in the sign-specialised dense kernel (verification loop inside the one-body form, own atan2 on x > 0)
    against the general-form kernel (bits 0 + 4: library atan2 at four corners): same algorithm, roundings differ by the
    pads, so the accumulators agree except at knife edges - on a full 14^5 grid, ragged shapes and an odd lambda grid."""
    rig = Rig(g.chamber_c1(), precision=precision, flags=RIG)
    try:
        ev = g.make_event(rig.ch, 31, n_noise=10)
        hd, oh = rig.hits(ev.wire, ev.drift)
        for dims in ((14,) * 5, (5, 4, 10, 19, 12), (3, 3, 6, 20, 7)):
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=RIG)
            vf = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=RIG | b.FLAG_GENERAL)
            vg = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, dims)
            rig.ctx.synchronize()
            vf, vg = vf.cpu().numpy(), vg.cpu().numpy()
            bad = np.nonzero(vf != vg)[0]
            assert len(bad) <= max(1, len(vf) // (100000 if precision == 64 else 2000)), (dims, len(bad), vf[bad[:10]], vg[bad[:10]])
            assert vf.max() > 0
    finally:
        rig.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_rigorous_refinement_children_kernel_matches_the_oracle(precision):
    """IA_FLAG_RIGOROUS_PHI in the sign-specialised CHILDREN kernel (round 2; before, a rigorous refinement took the general-form
    children kernel): kept boxes, votes and parameters of a batch refinement identical to the oracle's rigorous mode at
    every level, and to the general-form kernels (bits 0 + 4)."""
    rig = Rig(g.chamber_c1(), precision=precision, flags=RIG)
    try:
        evs = [g.make_event(rig.ch, 700 + e, n_noise=10) for e in range(6)]
        wire, drift = np.concatenate([e.wire for e in evs]), np.concatenate([e.drift for e in evs])
        off = np.cumsum([0] + [e.n_hits for e in evs]).astype(np.int32)
        hd, oh = rig.hits(wire, drift)
        od = rig.ctx.to_device(off)
        for levels, k in ((6, 8), (5, 16), (4, 3)):
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=RIG)
            boxes, par = rig.ctx.ia_refine_batch(hd, od, len(evs), 30, LO, HI, (8,) * 5, levels, k)
            rig.ctx.synchronize()
            gb = b.boxes_to_numpy(boxes, (len(evs), levels, k))
            ob, opar = o.refine_batch(rig.owires, oh, off, rig.oparams, LO, HI, (8,) * 5, levels, k)
            assert (gb["lo"] == ob["lo"]).all() and (gb["hi"] == ob["hi"]).all() and (gb["votes"] == ob["votes"]).all(), (levels, k)
            assert (par.cpu().numpy().reshape(opar.shape) == opar).all()
            rig.ctx.ia_set_params(g.TOL, precision=precision, flags=RIG | b.FLAG_GENERAL)
            boxes2, par2 = rig.ctx.ia_refine_batch(hd, od, len(evs), 30, LO, HI, (8,) * 5, levels, k)
            rig.ctx.synchronize()
            g2 = b.boxes_to_numpy(boxes2, (len(evs), levels, k))
            assert (gb["lo"] == g2["lo"]).all() and (gb["hi"] == g2["hi"]).all() and (gb["votes"] == g2["votes"]).all()
    finally:
        rig.close()
