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


def trace_mismatches(rig: Rig, hd, oh, blo, bhi, rel=1e-12):
    """G25: every vote mismatch must come from a (box, hit, sign) whose residual endpoint lies
    within `rel` (relative to the residual's scale) of zero on either side.  Returns the number of
    (box, hit) pairs that explain a mismatch; raises if a box has no such pair."""
    rg = rig.gpu_residual(hd, len(oh), blo, bhi)
    ro = o.residual(rig.owires, oh, rig.oparams, blo, bhi)
    explained = 0
    for i in range(len(blo)):
        ok = False
        for h in range(len(oh)):
            for s in range(2):
                for r in (rg[i, h, s], ro[i, h, s]):
                    if r[3]:
                        continue
                    if min(abs(r[0]), abs(r[1])) <= rel * r[2]:
                        ok = True
        if not ok:
            raise AssertionError(f"unexplained vote mismatch in box {i}: lo={blo[i]} hi={bhi[i]}")
        explained += 1
    return explained


def compare_votes(rig: Rig, hd, oh, vg: np.ndarray, vo: np.ndarray, boxes_of, min_equal=0.9999):
    """vg, vo: accumulators of the same cells.  boxes_of(indices) -> (blo, bhi) for tracing."""
    assert vg.shape == vo.shape
    bad = np.nonzero(vg != vo)[0]
    frac = 1.0 - len(bad) / max(len(vg), 1)
    assert frac >= min_equal, f"only {frac:.6f} of cells equal ({len(bad)} mismatches)"
    if len(bad):
        blo, bhi = boxes_of(bad[:200])
        trace_mismatches(rig, hd, oh, blo, bhi)
    return len(bad)
