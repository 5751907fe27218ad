"""ctypes binding of the oracle library (TEST INFRASTRUCTURE ONLY - see ia_oracle.cpp).

Argument marshalling only; every computation is in ia_oracle.cpp.  Arrays are numpy on the host.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

WIRE_DT = np.dtype([("x0", "f8"), ("y0", "f8"), ("sin_phi_s", "f8"), ("cos_phi_s", "f8"), ("tan_tau", "f8")])
HIT_DT = np.dtype([("wire", "i4"), ("pad", "i4"), ("drift", "f8")])
BOX_DT = np.dtype([("lo", "f8", (5,)), ("hi", "f8", (5,)), ("votes", "u2"), ("pad", "u2", (3,))])


class Params(C.Structure):
    _fields_ = [("tol", C.c_double), ("x_ref", C.c_double), ("y_ref", C.c_double), ("z_ref", C.c_double),
                ("precision", C.c_int32), ("flags", C.c_uint32)]


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        for name in ("orc_prim", "orc_residual", "orc_vote_boxes", "orc_vote", "orc_cell_boxes", "orc_topk",
                     "orc_refine", "orc_refine_batch", "orc_pad_ulps", "orc_max_threads", "orc_dax_point",
                     "orc_residual_paper", "orc_vote_paper", "orc_cell_boxes4", "orc_disk_filter",
                     "orc_select_max_paper", "orc_find_hits_paper", "orc_track_paper"):
            getattr(_lib, name).restype = C.c_int
        _lib.orc_set_threads.restype = None
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed: rc={rc}")


def make_params(tol, x_ref=0.0, y_ref=0.0, z_ref=0.0, precision=64, flags=0) -> Params:
    return Params(tol, x_ref, y_ref, z_ref, precision, flags)


def wires_of(chamber) -> np.ndarray:
    w = np.zeros(chamber.n_wires, WIRE_DT)
    w["x0"], w["y0"] = chamber.x0, chamber.y0
    w["sin_phi_s"], w["cos_phi_s"], w["tan_tau"] = chamber.sin_phi_s, chamber.cos_phi_s, chamber.tan_tau
    return w


def hits_of(wire_ids, drifts) -> np.ndarray:
    h = np.zeros(len(wire_ids), HIT_DT)
    h["wire"], h["drift"] = wire_ids, drifts
    return h


def set_threads(n: int):
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return lib().orc_max_threads()


def pad_ulps() -> int:
    return lib().orc_pad_ulps()


def prim(op: int, a, b=(0.0, 0.0), prec: int = 64):
    out = (C.c_double * 2)()
    _chk(lib().orc_prim(op, prec, C.c_double(a[0]), C.c_double(a[1]), C.c_double(b[0]), C.c_double(b[1]), out), "prim")
    return out[0], out[1]


def residual(wires, hits, params: Params, blo, bhi) -> np.ndarray:
    """f enclosures [n_boxes, n_hits, 2 signs (+,-), 4 = (f.lo, f.hi, scale, decided)]."""
    blo = np.ascontiguousarray(blo, np.float64).reshape(-1, 5)
    bhi = np.ascontiguousarray(bhi, np.float64).reshape(-1, 5)
    out = np.zeros((blo.shape[0], len(hits), 2, 4))
    _chk(lib().orc_residual(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), _p(blo), _p(bhi),
                            C.c_int64(blo.shape[0]), _p(out)), "residual")
    return out


def vote_boxes(wires, hits, params: Params, blo, bhi) -> np.ndarray:
    blo = np.ascontiguousarray(blo, np.float64).reshape(-1, 5)
    bhi = np.ascontiguousarray(bhi, np.float64).reshape(-1, 5)
    out = np.zeros(blo.shape[0], np.uint16)
    _chk(lib().orc_vote_boxes(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), _p(blo), _p(bhi),
                              C.c_int64(blo.shape[0]), _p(out)), "vote_boxes")
    return out


def vote(wires, hits, params: Params, lo, hi, dims, cell_idx=None) -> np.ndarray:
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    if cell_idx is None:
        n = int(np.prod(dims.astype(np.int64)))
        idx_p, n_idx = None, 0
    else:
        cell_idx = np.ascontiguousarray(cell_idx, np.int64)
        n = len(cell_idx)
        idx_p, n_idx = _p(cell_idx), n
    out = np.zeros(n, np.uint16)
    _chk(lib().orc_vote(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), _p(lo), _p(hi), _p(dims),
                        idx_p, C.c_int64(n_idx), _p(out)), "vote")
    return out


def cell_boxes(lo, hi, dims, cell_idx):
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    cell_idx = np.ascontiguousarray(cell_idx, np.int64)
    blo = np.zeros((len(cell_idx), 5))
    bhi = np.zeros((len(cell_idx), 5))
    _chk(lib().orc_cell_boxes(_p(lo), _p(hi), _p(dims), _p(cell_idx), C.c_int64(len(cell_idx)), _p(blo), _p(bhi)),
         "cell_boxes")
    return blo, bhi


def topk(votes, k: int):
    votes = np.ascontiguousarray(votes, np.uint16)
    idx = np.zeros(k, np.int64)
    v = np.zeros(k, np.uint16)
    _chk(lib().orc_topk(_p(votes), C.c_int64(len(votes)), k, _p(idx), _p(v)), "topk")
    return idx, v


def refine(wires, hits, params: Params, lo, hi, grid0, levels: int, k: int):
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    grid0 = np.ascontiguousarray(grid0, np.int32)
    boxes = np.zeros((levels, k), BOX_DT)
    par = np.zeros(20)          # centre[5], half-width[5] of the rank-0 box; hull lo[5], hi[5] of the kept boxes at the maximum (G19)
    _chk(lib().orc_refine(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), _p(lo), _p(hi), _p(grid0),
                          levels, k, _p(boxes), _p(par)), "refine")
    return boxes, par


def refine_batch(wires, hits, hit_offsets, params: Params, lo, hi, grid0, levels: int, k: int):
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    grid0 = np.ascontiguousarray(grid0, np.int32)
    hit_offsets = np.ascontiguousarray(hit_offsets, np.int32)
    n_ev = len(hit_offsets) - 1
    boxes = np.zeros((n_ev, levels, k), BOX_DT)
    par = np.zeros((n_ev, 20))
    _chk(lib().orc_refine_batch(_p(wires), len(wires), _p(hits), _p(hit_offsets), n_ev, C.byref(params), _p(lo),
                                _p(hi), _p(grid0), levels, k, _p(boxes), _p(par)), "refine_batch")
    return boxes, par


# ---- paper mode (ia_oracle.cpp "Paper-mode vote") --------------------------------------------
def dax_point(wire_row, params: Params, point, d_signed: float):
    """(ok, radicand of (A.5b), d_Ax) of steps S2-S8 at the point (xc, yc, R, z0, lambda), plain double."""
    w = np.zeros(1, WIRE_DT)
    w[0] = wire_row
    pt = np.ascontiguousarray(point, np.float64)
    out = np.zeros(2)
    rc = lib().orc_dax_point(_p(w), C.byref(params), _p(pt), C.c_double(d_signed), _p(out))
    if rc < 0:
        raise RuntimeError(f"oracle dax_point failed: rc={rc}")
    return rc == 0, out[0], out[1]


def residual_paper(wires, hits, params: Params, P: float, blo, bhi) -> np.ndarray:
    """condition (4) enclosures [n_boxes, n_hits, 2 lambda signs (+,-), 2 drift signs (+,-), 4 = (f.lo, f.hi, scale, has)]."""
    blo = np.ascontiguousarray(blo, np.float64).reshape(-1, 4)
    bhi = np.ascontiguousarray(bhi, np.float64).reshape(-1, 4)
    out = np.zeros((blo.shape[0], len(hits), 2, 2, 4))
    _chk(lib().orc_residual_paper(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), C.c_double(P), _p(blo),
                                  _p(bhi), C.c_int64(blo.shape[0]), _p(out)), "residual_paper")
    return out


def vote_paper(wires, hits, params: Params, P: float, lo, hi, dims, cell_idx=None, hit_mask=None, r_disk=-1.0) -> np.ndarray:
    """two 4-D accumulators [2, n]: [0] for lambda >= 0, [1] for lambda < 0; voxel index z0 fastest.
    hit_mask: uint8 per hit (0 = not used); r_disk >= 0: disk pre-filter (3a,b)."""
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    if cell_idx is None:
        n = int(np.prod(dims.astype(np.int64)))
        idx_p, n_idx = None, 0
    else:
        cell_idx = np.ascontiguousarray(cell_idx, np.int64)
        n = len(cell_idx)
        idx_p, n_idx = _p(cell_idx), n
    out = np.zeros((2, n), np.uint16)
    mask_p = None
    if hit_mask is not None:
        hit_mask = np.ascontiguousarray(hit_mask, np.uint8)
        mask_p = _p(hit_mask)
    _chk(lib().orc_vote_paper(_p(wires), len(wires), _p(hits), len(hits), mask_p, C.byref(params), C.c_double(P),
                              C.c_double(r_disk), _p(lo), _p(hi), _p(dims), idx_p, C.c_int64(n_idx), _p(out)), "vote_paper")
    return out


def cell_boxes4(lo, hi, dims, cell_idx):
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    cell_idx = np.ascontiguousarray(cell_idx, np.int64)
    blo = np.zeros((len(cell_idx), 4))
    bhi = np.zeros((len(cell_idx), 4))
    _chk(lib().orc_cell_boxes4(_p(lo), _p(hi), _p(dims), _p(cell_idx), C.c_int64(len(cell_idx)), _p(blo), _p(bhi)),
         "cell_boxes4")
    return blo, bhi


# ---- pieces of the paper's iteration scheme ------------------------------------------------------
class PaperFit(C.Structure):
    _fields_ = [("value", C.c_double * 4), ("error", C.c_double * 4), ("lam", C.c_double), ("lambda_sign", C.c_int32),
                ("vmax", C.c_int32), ("n_sel", C.c_int64), ("x_ref", C.c_double), ("y_ref", C.c_double), ("z0_centre", C.c_double)]


def disk_filter(lo, hi, dims, r_disk: float, cell_idx=None) -> np.ndarray:
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    if cell_idx is None:
        n, idx_p, n_idx = int(np.prod(dims.astype(np.int64))), None, 0
    else:
        cell_idx = np.ascontiguousarray(cell_idx, np.int64)
        n, idx_p, n_idx = len(cell_idx), _p(cell_idx), len(cell_idx)
    out = np.zeros(n, np.uint8)
    _chk(lib().orc_disk_filter(_p(lo), _p(hi), _p(dims), C.c_double(r_disk), idx_p, C.c_int64(n_idx), _p(out)), "disk_filter")
    return out


def select_max_paper(votes, lo, hi, dims, P: float, which: int = 0) -> PaperFit:
    votes = np.ascontiguousarray(votes, np.uint16)
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    dims = np.ascontiguousarray(dims, np.int32)
    fit = PaperFit()
    _chk(lib().orc_select_max_paper(_p(votes), _p(lo), _p(hi), _p(dims), C.c_double(P), int(which), C.byref(fit)), "select_max_paper")
    return fit


def find_hits_paper(wires, hits, params: Params, P: float, lambda_sign: int, lo, hi) -> np.ndarray:
    lo = np.ascontiguousarray(lo, np.float64)
    hi = np.ascontiguousarray(hi, np.float64)
    out = np.zeros(len(hits), np.uint8)
    _chk(lib().orc_find_hits_paper(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), C.c_double(P),
                                   int(lambda_sign), _p(lo), _p(hi), _p(out)), "find_hits_paper")
    return out


PASS_DT = np.dtype([("lo", "f8", (4,)), ("hi", "f8", (4,)), ("dims", "i4", (4,)), ("windowed", "i4"), ("move_ref", "i4")])
FIT_DT = np.dtype([("value", "f8", (4,)), ("error", "f8", (4,)), ("lam", "f8"), ("lambda_sign", "i4"), ("vmax", "i4"),
                   ("n_sel", "i8"), ("x_ref", "f8"), ("y_ref", "f8"), ("z0_centre", "f8")])


def make_passes(spec, move_ref=False) -> np.ndarray:
    """spec: list of ("grid", lo4, hi4, dims4) or ("window", half4, dims4); move_ref: every pass but the first is voted
    with the reference point of L98 (reading F2d')."""
    ps = np.zeros(len(spec), PASS_DT)
    ps["move_ref"][1:] = 1 if move_ref else 0
    for i, s in enumerate(spec):
        if s[0] == "grid":
            ps[i]["lo"], ps[i]["hi"], ps[i]["dims"], ps[i]["windowed"] = s[1], s[2], s[3], 0
        else:
            ps[i]["lo"], ps[i]["hi"], ps[i]["dims"], ps[i]["windowed"] = s[1], s[1], s[2], 1
    return ps


def move_ref_paper(wires, hits, mask, params: Params, prev_fit):
    """F2d' (L98): (index of the selected hit whose wire point in the plane z_ref is closest to the circle of prev_fit,
    or -1; the new reference point (x, y))."""
    out = np.zeros(2)
    fit = np.zeros(1, FIT_DT)
    fit[0] = prev_fit
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    rc = lib().orc_move_ref_paper(_p(wires), len(wires), _p(hits), len(hits), None if m is None else _p(m), C.byref(params),
                                  _p(fit), _p(out))
    if rc < -1:
        _chk(rc, "move_ref_paper")
    return rc, out


def transport_z0(params: Params, prev_fit, x_new: float, y_new: float) -> float:
    """z0 of prev_fit re-expressed for the reference point (x_new, y_new) (reading F2d')."""
    fit = np.zeros(1, FIT_DT)
    fit[0] = prev_fit
    f = lib().orc_transport_z0
    f.restype = C.c_double
    return float(f(C.byref(params), _p(fit), C.c_double(x_new), C.c_double(y_new)))


def track_paper(wires, hits, params: Params, P: float, r_disk: float, factor: float, passes: np.ndarray):
    """the paper's iteration scheme, one chain per sign of lambda: (fits [n_passes, 2] of FIT_DT, final sign)."""
    fits = np.zeros((len(passes), 2), FIT_DT)
    sign = C.c_int32(0)
    _chk(lib().orc_track_paper(_p(wires), len(wires), _p(hits), len(hits), C.byref(params), C.c_double(P), C.c_double(r_disk),
                               C.c_double(factor), _p(passes), len(passes), _p(fits), C.byref(sign)), "track_paper")
    return fits, int(sign.value)
