"""Shared plumbing for the -m gpu parity tests: one context per chamber, uploads, mismatch tracing."""
from __future__ import annotations

import numpy as np

from paper_2401_04576_b200 import binding as b
from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

LO, HI = np.array(g.BOX_LO), np.array(g.BOX_HI)


class Rig:
    """A chamber loaded on both sides."""

    def __init__(self, chamber, tol=g.TOL, precision=64, x_ref=0.0, y_ref=0.0, z_ref=0.0, flags=0):
        import torch
        self.torch = torch
        self.ch = chamber
        self.precision = precision
        self.ctx = b.Context(0)
        self.ctx.ia_load_geometry(b.wires_of(chamber))
        self.ctx.ia_set_params(tol, x_ref, y_ref, z_ref, precision, flags)
        self.owires = o.wires_of(chamber)
        self.oparams = o.make_params(tol, x_ref, y_ref, z_ref, precision, flags)

    def hits(self, wire, drift):
        """(device hits tensor, oracle hits array)"""
        return self.ctx.to_device(b.hits_of(wire, drift)), o.hits_of(wire, drift)

    def dev(self, a):
        return self.ctx.to_device(np.ascontiguousarray(a))

    def gpu_residual(self, hd, n_hits, blo, bhi):
        r = self.ctx.ia_residual(hd, n_hits, self.dev(blo), self.dev(bhi))
        self.ctx.synchronize()
        return r.cpu().numpy()

    def close(self):
        self.ctx.close()


def _bits(res):
    """per-(box, hit) vote bit from residual enclosures [box, hit, sign, (lo, hi, scale, forced)]: either sign cannot be excluded"""
    v = (res[..., 3] == 1) | ~((res[..., 0] > 0) | (res[..., 1] < 0))
    return v.any(axis=-1)


def gpu_hit_bits(rig: Rig, hd, n_hits, blo, bhi, kind):
    """Vote of every single hit for every box, through the kernel that produced the accumulator: kind "dense" = ia_vote
    with one hit on the one-cell grid [blo, bhi] (the sign-specialised dense kernel; cell edges of a one-cell grid are
    blo and bhi themselves, and the guards that pick its form can only relax on a sub-box), "boxes" = ia_vote_boxes."""
    bits = np.zeros((len(blo), n_hits), bool)
    ctx = rig.ctx
    if kind == "boxes":
        lo_d, hi_d = rig.dev(blo), rig.dev(bhi)
        for h in range(n_hits):
            bits[:, h] = ctx.ia_vote_boxes(hd[16 * h:16 * (h + 1)], 1, lo_d, hi_d).cpu().numpy() > 0
        return bits
    for i in range(len(blo)):
        for h in range(n_hits):
            bits[i, h] = int(ctx.ia_vote(hd[16 * h:16 * (h + 1)], 1, blo[i], bhi[i], (1,) * 5).cpu().numpy()[0]) > 0
    return bits


def trace_mismatches(rig: Rig, hd, oh, blo, bhi, vg=None, vo=None, rel=None, kind="dense"):
    """G25 as written: every vote mismatch is traced to the (box, hit) whose vote differs, and for THAT hit an endpoint of
    the residual enclosure of one of its drift signs (the oracle's orc_residual or the GPU's ia_residual) must lie within
    `rel` (relative to the residual's scale; 1e-12 in FP64, 2^-18 in FP32: G22) of zero.  The per-hit votes are read from
    the kernel that made the accumulator (gpu_hit_bits) and from the oracle's enclosures; when vg / vo (the two vote counts
    of the boxes) are given, the per-hit votes must add up to them.  Returns the number of (box, hit) pairs traced."""
    n_hits = len(oh)
    if rel is None:
        rel = 1e-12 if rig.precision == 64 else 2.0 ** -18
    rg = rig.gpu_residual(hd, n_hits, blo, bhi)
    ro = o.residual(rig.owires, oh, rig.oparams, blo, bhi)
    bg = gpu_hit_bits(rig, hd, n_hits, blo, bhi, kind)
    bo = _bits(ro)
    if vg is not None:
        assert (bg.sum(axis=1) == vg).all(), "per-hit GPU votes do not add up to the accumulator"
    if vo is not None:
        assert (bo.sum(axis=1) == vo).all(), "per-hit oracle votes do not add up to the oracle's accumulator"

    def knife(r):              # [sign, 4] -> an endpoint of either sign within the band
        return any((not r[s, 3]) and min(abs(r[s, 0]), abs(r[s, 1])) <= rel * r[s, 2] for s in range(2))

    traced = 0
    for i, h in np.argwhere(bg != bo):
        if not (knife(ro[i, h]) or knife(rg[i, h])):
            raise AssertionError(f"unexplained vote mismatch: box {i} lo={blo[i]} hi={bhi[i]} hit {h}: gpu votes {bg[i, h]}, "
                                 f"oracle {bo[i, h]}; oracle f = {ro[i, h, :, :3].tolist()}, gpu f = {rg[i, h, :, :3].tolist()}")
        traced += 1
    if vg is not None and vo is not None:
        assert (bg != bo).any(axis=1)[np.asarray(vg) != np.asarray(vo)].all()
    return traced


def compare_votes(rig: Rig, hd, oh, vg: np.ndarray, vo: np.ndarray, boxes_of, min_equal=0.9999, kind="dense"):
    """vg, vo: accumulators of the same cells.  boxes_of(indices) -> (blo, bhi) for tracing.  The bar is north_star's:
    >= 99.99 % of the cells equal and every mismatch traced (at most 200 of them are traced per call)."""
    assert vg.shape == vo.shape
    bad = np.nonzero(vg != vo)[0]
    frac = 1.0 - len(bad) / max(len(vg), 1)
    assert frac >= min_equal, f"only {frac:.6f} of cells equal ({len(bad)} mismatches)"
    if len(bad):
        blo, bhi = boxes_of(bad[:200])
        trace_mismatches(rig, hd, oh, blo, bhi, vg[bad[:200]], vo[bad[:200]], kind=kind)
    return len(bad)
