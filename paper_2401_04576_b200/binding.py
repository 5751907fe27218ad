"""Thin ctypes binding of libia_b200.so (include/ia.h).  Argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module converts torch
tensors to device pointers, host numpy arrays to host pointers, and error codes to exceptions.
There is no CPU fallback: if the library is missing or fails, the call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libia_b200.so")

IA_MAX_HITS = 1024
IA_MAX_K = 32
IA_N_PARAMS = 20

WIRE_DT = np.dtype([("x0", "f8"), ("y0", "f8"), ("sin_phi_s", "f8"), ("cos_phi_s", "f8"), ("tan_tau", "f8"),
                    ("half_len", "f8"), ("layer", "i4"), ("_pad", "i4")])
HIT_DT = np.dtype([("wire", "i4"), ("_pad", "i4"), ("drift", "f8")])
BOX_DT = np.dtype([("lo", "f8", (5,)), ("hi", "f8", (5,)), ("votes", "u2"), ("_pad", "u2", (3,))])
FIT_DT = np.dtype([("value", "f8", (4,)), ("error", "f8", (4,)), ("lam", "f8"), ("lambda_sign", "i4"), ("vmax", "i4"),
                   ("n_sel", "i8"), ("x_ref", "f8"), ("y_ref", "f8"), ("z0_centre", "f8")])
PASS_DT = np.dtype([("lo", "f8", (4,)), ("hi", "f8", (4,)), ("dims", "i4", (4,)), ("windowed", "i4"), ("move_ref", "i4")])
assert WIRE_DT.itemsize == 56 and HIT_DT.itemsize == 16 and BOX_DT.itemsize == 88 and FIT_DT.itemsize == 112

EXPORTS = ("ia_create", "ia_destroy", "ia_load_geometry", "ia_set_params", "ia_vote", "ia_vote_slab", "ia_topk_keys", "ia_merge_keys", "ia_vote_boxes", "ia_vote_paper", "ia_select_max_paper", "ia_find_hits_paper", "ia_track_paper", "ia_topk",
           "ia_topk_static", "ia_topk_static_error", "ia_set_host_slab_min",
           "ia_refine", "ia_refine_batch", "ia_vote_host", "ia_refine_batch_host", "ia_residual", "ia_residual_fast", "ia_prim",
           "ia_probe_fp64", "ia_device_status", "ia_launch_count", "ia_graph_replays", "ia_strerror", "ia_last_cuda_error", "ia_pad_ulps")

KEY_LIST = 32      # IA_KEY_LIST
# IA_FLAG_* of include/ia.h (bits of ia_params.flags)
FLAG_GENERAL, FLAG_ONE_BODY, FLAG_THREE_BODY, FLAG_FULL_TURN = 1, 2, 4, 8
FLAG_RIGOROUS_PHI, FLAG_NO_GRAPH, FLAG_PREFILTER, FLAG_NO_PDL = 16, 32, 64, 128


class IaParams(C.Structure):
    _fields_ = [("tol", C.c_double), ("x_ref", C.c_double), ("y_ref", C.c_double), ("z_ref", C.c_double),
                ("precision", C.c_int32), ("flags", C.c_uint32)]


class IaError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__(f"{what}: {detail} (code {code})")


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen libia_b200.so and declare the prototypes.  Raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(
            f"{path} not found: build it with `python -m paper_2401_04576_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    lib.ia_create.argtypes = [C.POINTER(vp), i32, vp]
    lib.ia_destroy.argtypes = [vp]
    lib.ia_destroy.restype = None
    lib.ia_load_geometry.argtypes = [vp, vp, i32]
    lib.ia_set_params.argtypes = [vp, C.POINTER(IaParams)]
    lib.ia_vote.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    lib.ia_vote_boxes.argtypes = [vp, vp, i32, vp, vp, i64, vp]
    lib.ia_vote_slab.argtypes = [vp, vp, i32, vp, vp, vp, i32, i32, vp]
    lib.ia_topk_keys.argtypes = [vp, vp, i64, i32, i64, vp]
    lib.ia_merge_keys.argtypes = [vp, vp, i32, i32, vp, vp]
    lib.ia_vote_paper.argtypes = [vp, vp, i32, vp, dbl, dbl, vp, vp, vp, vp]
    lib.ia_select_max_paper.argtypes = [vp, vp, dbl, vp, vp, vp, i32, vp]
    lib.ia_track_paper.argtypes = [vp, vp, i32, dbl, dbl, dbl, vp, i32, vp, vp]
    lib.ia_find_hits_paper.argtypes = [vp, vp, i32, dbl, vp, dbl, vp]
    lib.ia_topk.argtypes = [vp, vp, i64, i32, vp, vp]
    lib.ia_topk_static.argtypes = [i32, vp, vp, i64, i32, vp, vp]
    lib.ia_topk_static_error.argtypes = []
    lib.ia_topk_static_error.restype = C.c_char_p
    lib.ia_refine.argtypes = [vp, vp, i32, vp, vp, vp, i32, i32, vp, vp]
    lib.ia_refine_batch.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp, i32, i32, vp, vp]
    lib.ia_vote_host.argtypes = [vp, vp, i32, vp, vp, vp, vp]
    lib.ia_refine_batch_host.argtypes = [vp, vp, vp, i32, vp, vp, vp, i32, i32, vp, vp]
    lib.ia_set_host_slab_min.argtypes = [vp, i64]
    lib.ia_residual.argtypes = [vp, vp, i32, vp, vp, i64, vp]
    lib.ia_residual_fast.argtypes = [vp, vp, i32, vp, vp, i64, vp]
    lib.ia_prim.argtypes = [vp, i32, i32, vp, vp, i64, vp]
    lib.ia_probe_fp64.argtypes = [vp, i32, i32, i32, vp]
    lib.ia_device_status.argtypes = [vp]
    lib.ia_launch_count.argtypes = [vp]
    lib.ia_launch_count.restype = i64
    lib.ia_graph_replays.argtypes = [vp]
    lib.ia_graph_replays.restype = i64
    lib.ia_strerror.argtypes = [i32]
    lib.ia_strerror.restype = C.c_char_p
    lib.ia_last_cuda_error.argtypes = [vp]
    lib.ia_last_cuda_error.restype = C.c_char_p
    lib.ia_pad_ulps.argtypes = []
    _lib = lib
    return lib


TOPK_STATIC_LISTS = 1024                 # IA_TOPK_STATIC_LISTS
TOPK_STATIC_MAX_CELLS = 1 << 40          # IA_TOPK_STATIC_MAX_CELLS


def ia_topk_static(votes_dev, k, idx_out, votes_out, n_cells=None, stream=None):
    """ia_topk for callers that must not allocate on the device (see include/ia.h): no context, no torch allocation -
    the caller owns the accumulator and both outputs (idx_out: int64[k], votes_out: uint16[k], CUDA tensors on the
    accumulator's device), the work is enqueued on `stream` (default: torch's current stream of that device) and the
    candidate lists live in the library's fixed 256 KB device array.  Calls on one GPU must not overlap."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("libia_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    dev = votes_dev.device.index
    if idx_out.dtype != torch.int64 or votes_out.dtype != torch.uint16 or idx_out.numel() < k or votes_out.numel() < k:
        raise ValueError("idx_out must be int64[k] and votes_out uint16[k]")
    if idx_out.device != votes_dev.device or votes_out.device != votes_dev.device:
        raise ValueError("outputs must live on the accumulator's device")
    n = votes_dev.numel() if n_cells is None else int(n_cells)
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    rc = lib.ia_topk_static(dev, C.c_void_p(s.cuda_stream), _dp(votes_dev), n, int(k), _dp(idx_out), _dp(votes_out))
    if rc != 0:
        raise IaError(rc, "ia_topk_static", lib.ia_topk_static_error().decode())
    return idx_out, votes_out


def wires_of(chamber) -> np.ndarray:
    """eventgen.Chamber -> ia_wire[] (host)."""
    w = np.zeros(chamber.n_wires, WIRE_DT)
    w["x0"], w["y0"] = chamber.x0, chamber.y0
    w["sin_phi_s"], w["cos_phi_s"], w["tan_tau"] = chamber.sin_phi_s, chamber.cos_phi_s, chamber.tan_tau
    w["half_len"], w["layer"] = chamber.half_len, chamber.layer
    return w


def hits_of(wire_ids, drifts) -> np.ndarray:
    h = np.zeros(len(wire_ids), HIT_DT)
    h["wire"], h["drift"] = wire_ids, drifts
    return h


def _host5(a, dtype):
    a = np.ascontiguousarray(a, dtype)
    if a.shape != (5,):
        raise ValueError("expected 5 values (xc, yc, R, z0, lambda)")
    return a


def _host4(a, dtype):
    a = np.ascontiguousarray(a, dtype)
    if a.shape != (4,):
        raise ValueError("expected 4 values (xc, yc, R, z0)")
    return a


def _hp(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dp(t):
    """device pointer of a contiguous CUDA torch tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


class Context:
    """ia_ctx: geometry + parameters + stream.  Same names as the C ABI."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        self._torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("libia_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = device
        torch.cuda.set_device(device)
        torch.cuda.init()
        torch.zeros(1, device=f"cuda:{device}")            # make sure the primary context exists
        self.stream = stream if stream is not None else torch.cuda.current_stream(device)
        h = C.c_void_p()
        self._chk(self.lib.ia_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream)), "ia_create", None)
        self.h = h
        self.n_wires = 0

    def _chk(self, rc: int, what: str, h="self"):
        if rc == 0:
            return
        detail = self.lib.ia_strerror(rc).decode()
        if rc == -5 and h is not None:
            detail += ": " + self.lib.ia_last_cuda_error(self.h).decode()
        raise IaError(rc, what, detail)

    def close(self):
        if getattr(self, "h", None):
            self.lib.ia_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- a1
    def ia_load_geometry(self, wires: np.ndarray):
        wires = np.ascontiguousarray(wires, WIRE_DT)
        self._chk(self.lib.ia_load_geometry(self.h, _hp(wires), len(wires)), "ia_load_geometry")
        self.n_wires = len(wires)

    def ia_set_params(self, tol=0.045, x_ref=0.0, y_ref=0.0, z_ref=0.0, precision=64, flags=0):
        p = IaParams(tol, x_ref, y_ref, z_ref, precision, flags)
        self._chk(self.lib.ia_set_params(self.h, C.byref(p)), "ia_set_params")

    def to_device(self, a: np.ndarray):
        """host structured/plain array -> CUDA uint8/typed tensor (plumbing for tests and bench)."""
        torch = self._torch
        a = np.ascontiguousarray(a)
        if a.dtype.fields is not None:
            t = torch.from_numpy(a.view(np.uint8).reshape(-1).copy())
        else:
            t = torch.from_numpy(a.copy())
        return t.to(f"cuda:{self.device}")

    def _empty(self, n, dtype):
        return self._torch.empty(int(n), dtype=dtype, device=f"cuda:{self.device}")

    # ---- a2-a6
    def ia_vote(self, hits_dev, n_hits, box_lo, box_hi, grid_dims, votes_out=None):
        torch = self._torch
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid_dims, np.int32)
        n = int(np.prod(dims.astype(np.int64)))
        if votes_out is None:
            votes_out = self._empty(n, torch.uint16)
        self._chk(self.lib.ia_vote(self.h, _dp(hits_dev), n_hits, _hp(lo), _hp(hi), _hp(dims), _dp(votes_out)), "ia_vote")
        return votes_out

    # ---- (e): the dense vote of the xc cells [ix_begin, ix_end) only, and the key lists that cross GPUs
    def ia_vote_slab(self, hits_dev, n_hits, box_lo, box_hi, grid_dims, ix_begin, ix_end, votes_out=None):
        torch = self._torch
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid_dims, np.int32)
        n = int(ix_end - ix_begin) * int(np.prod(dims[1:].astype(np.int64)))
        if votes_out is None:
            votes_out = self._empty(max(n, 0), torch.uint16)
        self._chk(self.lib.ia_vote_slab(self.h, _dp(hits_dev), n_hits, _hp(lo), _hp(hi), _hp(dims), int(ix_begin), int(ix_end),
                                        _dp(votes_out)), "ia_vote_slab")
        return votes_out

    def ia_topk_keys(self, votes_dev, k, index_base=0, n_cells=None, keys_out=None):
        torch = self._torch
        n = votes_dev.numel() if n_cells is None else n_cells
        if keys_out is None:
            keys_out = self._empty(KEY_LIST, torch.int64)          # uint64 keys carried as int64 bit patterns
        self._chk(self.lib.ia_topk_keys(self.h, _dp(votes_dev), n, k, int(index_base), _dp(keys_out)), "ia_topk_keys")
        return keys_out

    def ia_merge_keys(self, keys_dev, n_lists, k):
        torch = self._torch
        idx = self._empty(max(k, 1), torch.int64)
        v = self._empty(max(k, 1), torch.uint16)
        self._chk(self.lib.ia_merge_keys(self.h, _dp(keys_dev), int(n_lists), k, _dp(idx), _dp(v)), "ia_merge_keys")
        return idx, v

    # ---- f1: the paper's own configuration (4-D voxels, mid-voxel d_Ax, two lambda-sign accumulators)
    def ia_vote_paper(self, hits_dev, n_hits, momentum_radius, box_lo, box_hi, grid_dims, votes_out=None, hit_mask_dev=None,
                      r_disk=-1.0):
        torch = self._torch
        lo, hi, dims = _host4(box_lo, np.float64), _host4(box_hi, np.float64), _host4(grid_dims, np.int32)
        n = int(np.prod(dims.astype(np.int64)))
        if votes_out is None:
            votes_out = self._empty(2 * n, torch.uint16)
        self._chk(self.lib.ia_vote_paper(self.h, _dp(hits_dev), n_hits, _dp(hit_mask_dev), float(momentum_radius), float(r_disk),
                                         _hp(lo), _hp(hi), _hp(dims), _dp(votes_out)), "ia_vote_paper")
        return votes_out.view(2, n)

    # ---- f2 pieces: maximum-vote selection (device-resident result) and hit finding
    def ia_select_max_paper(self, votes_dev, momentum_radius, box_lo, box_hi, grid_dims, fit_out=None, which=0):
        torch = self._torch
        lo, hi, dims = _host4(box_lo, np.float64), _host4(box_hi, np.float64), _host4(grid_dims, np.int32)
        if fit_out is None:
            fit_out = self._empty(FIT_DT.itemsize, torch.uint8)
        self._chk(self.lib.ia_select_max_paper(self.h, _dp(votes_dev), float(momentum_radius), _hp(lo), _hp(hi), _hp(dims),
                                               int(which), _dp(fit_out)), "ia_select_max_paper")
        return fit_out

    def ia_track_paper(self, hits_dev, n_hits, momentum_radius, passes: np.ndarray, r_disk=10.0, factor=5.0, fits_out=None,
                       sign_out=None):
        """passes: PASS_DT array (host).  Returns (fits uint8 tensor holding [n_passes][2] FIT_DT, sign int32 tensor),
        both on the device; nothing is synchronised."""
        torch = self._torch
        passes = np.ascontiguousarray(passes, PASS_DT)
        if fits_out is None:
            fits_out = self._empty(2 * len(passes) * FIT_DT.itemsize, torch.uint8)
        if sign_out is None:
            sign_out = self._empty(1, torch.int32)
        self._chk(self.lib.ia_track_paper(self.h, _dp(hits_dev), n_hits, float(momentum_radius), float(r_disk), float(factor),
                                          _hp(passes), len(passes), _dp(fits_out), _dp(sign_out)), "ia_track_paper")
        return fits_out, sign_out

    def ia_find_hits_paper(self, hits_dev, n_hits, momentum_radius, fit_dev, factor=5.0, flags_out=None):
        torch = self._torch
        if flags_out is None:
            flags_out = self._empty(max(n_hits, 1), torch.uint8)
        self._chk(self.lib.ia_find_hits_paper(self.h, _dp(hits_dev), n_hits, float(momentum_radius), _dp(fit_dev), float(factor),
                                              _dp(flags_out)), "ia_find_hits_paper")
        return flags_out[:n_hits]

    def ia_vote_boxes(self, hits_dev, n_hits, lo_dev, hi_dev, votes_out=None):
        torch = self._torch
        n = lo_dev.numel() // 5
        if votes_out is None:
            votes_out = self._empty(n, torch.uint16)
        self._chk(self.lib.ia_vote_boxes(self.h, _dp(hits_dev), n_hits, _dp(lo_dev), _dp(hi_dev), n, _dp(votes_out)),
                  "ia_vote_boxes")
        return votes_out

    # ---- a7
    def ia_topk(self, votes_dev, k, n_cells=None):
        torch = self._torch
        n = votes_dev.numel() if n_cells is None else n_cells
        idx = self._empty(max(k, 1), torch.int64)
        v = self._empty(max(k, 1), torch.uint16)
        self._chk(self.lib.ia_topk(self.h, _dp(votes_dev), n, k, _dp(idx), _dp(v)), "ia_topk")
        return idx, v

    # ---- a8-a10
    def ia_refine(self, hits_dev, n_hits, box_lo, box_hi, grid0, levels, k, boxes=None, params=None):
        torch = self._torch
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid0, np.int32)
        if boxes is None:
            boxes = self._empty(max(levels * k, 1) * BOX_DT.itemsize, torch.uint8)
        if params is None:
            params = self._empty(IA_N_PARAMS, torch.float64)
        self._chk(self.lib.ia_refine(self.h, _dp(hits_dev), n_hits, _hp(lo), _hp(hi), _hp(dims), levels, k, _dp(boxes),
                                     _dp(params)), "ia_refine")
        return boxes, params

    def ia_refine_batch(self, hits_dev, hit_offsets_dev, n_events, max_hits, box_lo, box_hi, grid0, levels, k,
                        boxes=None, params=None):
        torch = self._torch
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid0, np.int32)
        if boxes is None:
            boxes = self._empty(max(n_events * levels * k, 1) * BOX_DT.itemsize, torch.uint8)
        if params is None:
            params = self._empty(max(n_events, 1) * IA_N_PARAMS, torch.float64)
        self._chk(self.lib.ia_refine_batch(self.h, _dp(hits_dev), _dp(hit_offsets_dev), n_events, max_hits, _hp(lo),
                                           _hp(hi), _hp(dims), levels, k, _dp(boxes), _dp(params)), "ia_refine_batch")
        return boxes, params

    # ---- host-buffer (end-to-end) variants
    def ia_vote_host(self, hits: np.ndarray, box_lo, box_hi, grid_dims, votes_out: np.ndarray | None = None):
        hits = np.ascontiguousarray(hits, HIT_DT)
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid_dims, np.int32)
        n = int(np.prod(dims.astype(np.int64)))
        if votes_out is None:
            votes_out = np.empty(n, np.uint16)
        self._chk(self.lib.ia_vote_host(self.h, _hp(hits), len(hits), _hp(lo), _hp(hi), _hp(dims), _hp(votes_out)),
                  "ia_vote_host")
        return votes_out

    def ia_set_host_slab_min(self, min_cells: int):
        self._chk(self.lib.ia_set_host_slab_min(self.h, int(min_cells)), "ia_set_host_slab_min")

    def ia_refine_batch_host(self, hits: np.ndarray, hit_offsets: np.ndarray, box_lo, box_hi, grid0, levels, k,
                             boxes: np.ndarray | None = None, params: np.ndarray | None = None):
        hits = np.ascontiguousarray(hits, HIT_DT)
        off = np.ascontiguousarray(hit_offsets, np.int32)
        n_events = len(off) - 1
        lo, hi, dims = _host5(box_lo, np.float64), _host5(box_hi, np.float64), _host5(grid0, np.int32)
        if boxes is None:
            boxes = np.zeros((n_events, levels, k), BOX_DT)
        if params is None:
            params = np.zeros((n_events, IA_N_PARAMS))
        self._chk(self.lib.ia_refine_batch_host(self.h, _hp(hits), _hp(off), n_events, _hp(lo), _hp(hi), _hp(dims), levels,
                                                k, _hp(boxes), _hp(params)), "ia_refine_batch_host")
        return boxes, params

    # ---- diagnostics
    def ia_residual(self, hits_dev, n_hits, lo_dev, hi_dev):
        torch = self._torch
        n = lo_dev.numel() // 5
        out = self._empty(n * n_hits * 2 * 4, torch.float64)
        self._chk(self.lib.ia_residual(self.h, _dp(hits_dev), n_hits, _dp(lo_dev), _dp(hi_dev), n, _dp(out)), "ia_residual")
        return out.view(n, n_hits, 2, 4)

    def ia_residual_fast(self, hits_dev, n_hits, lo_dev, hi_dev):
        torch = self._torch
        n = lo_dev.numel() // 5
        out = self._empty(n * n_hits * 2 * 4, torch.float64)
        self._chk(self.lib.ia_residual_fast(self.h, _dp(hits_dev), n_hits, _dp(lo_dev), _dp(hi_dev), n, _dp(out)), "ia_residual_fast")
        return out.view(n, n_hits, 2, 4)

    def ia_prim(self, op, prec, a_dev, b_dev=None):
        torch = self._torch
        n = a_dev.numel() // 2
        out = self._empty(2 * n, torch.float64)
        self._chk(self.lib.ia_prim(self.h, op, prec, _dp(a_dev), _dp(b_dev), n, _dp(out)), "ia_prim")
        return out.view(n, 2)

    def ia_probe_fp64(self, mode: int, iters: int, blocks: int) -> float:
        """FP64 thread-instructions per second sustained by independent chains (timed with CUDA events)."""
        torch = self._torch
        sink = self._empty(1, torch.float64)
        with torch.cuda.stream(self.stream):
            self._chk(self.lib.ia_probe_fp64(self.h, mode, iters, blocks, _dp(sink)), "ia_probe_fp64")   # warm-up
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record(self.stream)
            self._chk(self.lib.ia_probe_fp64(self.h, mode, iters, blocks, _dp(sink)), "ia_probe_fp64")
            t1.record(self.stream)
        t1.synchronize()
        return blocks * 256.0 * 8.0 * iters / (t0.elapsed_time(t1) * 1e-3)

    def ia_device_status(self):
        self._chk(self.lib.ia_device_status(self.h), "ia_device_status")

    def ia_launch_count(self) -> int:
        return int(self.lib.ia_launch_count(self.h))

    def ia_graph_replays(self) -> int:
        return int(self.lib.ia_graph_replays(self.h))

    def synchronize(self):
        self.stream.synchronize()


def boxes_to_numpy(boxes_u8, shape) -> np.ndarray:
    """uint8 CUDA tensor of ia_box records -> structured numpy array of the given shape."""
    return boxes_u8.cpu().numpy().view(BOX_DT).reshape(shape)
