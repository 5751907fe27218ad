"""-m gpu: parity at BASELINE.json's full sizes, in the launch configuration bench.py times (SURVEY 8(d) "Parity protocol").

  C1  every one of the 32^5 cells x 40 hits against the oracle, top-10 identical
  C3  all 1,024 events, FP64 and FP32 intervals: the kept boxes of all 8 passes, their votes and the parameters
      bit-identical to orc_refine_batch (north_star clause 1)
  C4  a stratified sample of the 64^5 grid: more than 2^24 distinct uniformly drawn cells (the floor SURVEY 8(d) sets), the GPU's top-10 cells, the truth cell and two
      complete (R, z0, lambda) columns (the truth's and a random one)

The oracle runs on the host cores (about a minute each on 16 cores), so these are the slow tests of the suite; every
vote mismatch is traced per hit (G25, gpu_common.trace_mismatches).
"""
import numpy as np
import pytest

from paper_2401_04576_b200 import binding as b
from paper_2401_04576_b200 import eventgen as g
from oracle import oracle as o

from gpu_common import HI, LO, Rig, compare_votes

pytestmark = pytest.mark.gpu


def _dense(cfg_idx, sample):
    cfg = g.config(cfg_idx)
    ev = cfg.events[0]
    rig = Rig(cfg.chamber)
    try:
        hd, oh = rig.hits(ev.wire, ev.drift)
        # the prefiltered kernel (IA_FLAG_PREFILTER) must give the brute-force accumulator bit for bit, at full size
        rig.ctx.ia_set_params(g.TOL, flags=b.FLAG_PREFILTER)
        votes_pf = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, cfg.grid)
        rig.ctx.ia_set_params(g.TOL, flags=0)
        votes = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, cfg.grid)
        idx, vv = rig.ctx.ia_topk(votes, 10)
        rig.ctx.synchronize()
        vg = votes.cpu().numpy()
        vpf = votes_pf.cpu().numpy()
        assert (vg == vpf).all(), f"prefilter changed {int((vg != vpf).sum())} cells"
        del votes_pf, vpf
        idx, vv = idx.cpu().numpy(), vv.cpu().numpy()
        n = vg.size
        truth = g.truth_cell(ev.track.params, LO, HI, cfg.grid)
        if sample is None:
            cells = None
            vo = o.vote(rig.owires, oh, rig.oparams, LO, HI, cfg.grid)
            vgs = vg
            oi, ov = o.topk(vo, 10)
            assert (oi == idx).all() and (ov == vv).all(), "top-10 of the oracle's accumulator differs from the GPU's"
        else:
            rng = np.random.default_rng(2024)
            col = int(np.prod(cfg.grid[2:]))
            cols = [truth // col, int(rng.integers(n // col))]
            extra = np.concatenate([idx, [truth]] + [np.arange(c * col, (c + 1) * col) for c in cols])
            cells = np.unique(np.concatenate([rng.integers(0, n, size=sample), extra])).astype(np.int64)
            vo = o.vote(rig.owires, oh, rig.oparams, LO, HI, cfg.grid, cell_idx=cells)
            vgs = vg[cells]
            # the GPU's top-10 is the exact top-10 of its own accumulator, and the oracle agrees on those cells' counts
            ei, evv = o.topk(vg, 10)
            assert (ei == idx).all() and (evv == vv).all()
            assert (vo[np.searchsorted(cells, idx)] == vv).all()
        where = (lambda i: o.cell_boxes(LO, HI, cfg.grid, i)) if cells is None else (lambda i: o.cell_boxes(LO, HI, cfg.grid, cells[i]))
        n_bad = compare_votes(rig, hd, oh, vgs, vo, where)
        assert vg.max() <= ev.n_hits
        return n_bad, vo.size, int(vg[truth])
    finally:
        rig.close()


def test_c1_every_cell():
    n_bad, n, _ = _dense(1, None)
    assert n == 32 ** 5 and n_bad <= n // 10000


def test_c4_stratified_sample():
    # ">= 2^24 cells incl. the top-10, the truth cell and two complete (R, z0, lambda) columns"; 2^24 + 2^19
    # draws with replacement leave more than 2^24 distinct cells (about 2^17 collisions are expected)
    n_bad, n, v_truth = _dense(4, (1 << 24) + (1 << 19))
    assert n >= (1 << 24) and n_bad <= n // 10000
    assert v_truth >= 38            # 40 genuine hits, 3-sigma tolerance on smeared drifts


@pytest.mark.slow
def test_c4_every_cell():
    """"C4 full if <= 1 h": every one of the 64^5 = 1,073,741,824 cells x 60 hits of the configuration the
    headline is quoted on (condition (4)), GPU accumulator against the oracle's, slab of xc cells by slab
    (64 slabs of 2^24 cells; about 50 s of oracle time each on 16 cores).  Run once per round, not by default:

        IA_RUN_SLOW=1 python -m pytest tests/test_gpu_fullsize.py -q -m gpu -k c4_every_cell

    Progress and the final counts are written to gpurun_out/c4_full_parity.json after every slab (a run cut short still
    leaves what it compared); BASELINE.md section 3 records the result."""
    import json
    import os
    import time
    cfg = g.config(4)
    ev = cfg.events[0]
    rig = Rig(cfg.chamber)
    out_dir = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(out_dir, exist_ok=True)
    try:
        hd, oh = rig.hits(ev.wire, ev.drift)
        votes = rig.ctx.ia_vote(hd, ev.n_hits, LO, HI, cfg.grid)
        rig.ctx.synchronize()
        vg = votes.cpu().numpy()
        n = vg.size
        nx = cfg.grid[0]
        per = n // nx
        done = {"config": "C4 64^5 x 60 hits, seed 4", "cells_total": n, "cells_compared": 0, "mismatches": 0, "traced": 0,
                "slabs_done": 0, "oracle_seconds": 0.0, "complete": False}
        for ix in range(nx):
            cells = np.arange(ix * per, (ix + 1) * per, dtype=np.int64)
            t0 = time.perf_counter()
            vo = o.vote(rig.owires, oh, rig.oparams, LO, HI, cfg.grid, cell_idx=cells)
            done["oracle_seconds"] += time.perf_counter() - t0
            n_bad = compare_votes(rig, hd, oh, vg[ix * per:(ix + 1) * per], vo, lambda i: o.cell_boxes(LO, HI, cfg.grid, cells[i]))
            done["cells_compared"] += per
            done["mismatches"] += int(n_bad)
            done["traced"] += int(min(n_bad, 200))          # compare_votes traces up to 200 per call and fails on an unexplained one
            done["slabs_done"] = ix + 1
            with open(os.path.join(out_dir, "c4_full_parity.json"), "w") as f:
                json.dump(done, f)
        done["complete"] = True
        with open(os.path.join(out_dir, "c4_full_parity.json"), "w") as f:
            json.dump(done, f)
        assert done["cells_compared"] == n and done["mismatches"] <= n // 10000
    finally:
        rig.close()


@pytest.mark.parametrize("precision", [64, 32])
def test_c3_all_1024_events_identical(precision):
    n_events = 1024
    cfg = g.config(3, n_events=n_events)
    rig = Rig(cfg.chamber, precision=precision)
    try:
        wire = np.concatenate([e.wire for e in cfg.events])
        drift = np.concatenate([e.drift for e in cfg.events])
        off = np.cumsum([0] + [e.n_hits for e in cfg.events]).astype(np.int32)
        hd, oh = rig.hits(wire, drift)
        boxes, par = rig.ctx.ia_refine_batch(hd, rig.dev(off), n_events, 30, LO, HI, cfg.grid, cfg.levels, cfg.k)
        rig.ctx.synchronize()
        gb = b.boxes_to_numpy(boxes, (n_events, cfg.levels, cfg.k))
        ob, opar = o.refine_batch(rig.owires, oh, off, rig.oparams, LO, HI, cfg.grid, cfg.levels, cfg.k)
        same = [(gb["lo"][e] == ob["lo"][e]).all() and (gb["hi"][e] == ob["hi"][e]).all() and (gb["votes"][e] == ob["votes"][e]).all()
                for e in range(n_events)]
        bad = [e for e in range(n_events) if not same[e]]
        assert not bad, f"events whose kept boxes differ from the oracle's: {bad[:20]}"
        assert (par.cpu().numpy().reshape(-1, 20) == opar).all()
    finally:
        rig.close()
