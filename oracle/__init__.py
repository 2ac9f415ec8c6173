"""ctypes binding of the CPU oracle (oracle/ffpp_oracle.cpp) — TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this.  It imports nothing from the CUDA package and the CUDA package imports nothing from here.
Marshalling only: every number is computed in ffpp_oracle.cpp.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ffpp_oracle.cpp")
_LIB = os.path.join(_HERE, "libffpp_oracle.so")


class OracleParams(ctypes.Structure):
    _fields_ = [
        ("dtype", ctypes.c_int32), ("conf_thresh", ctypes.c_float), ("iou_thresh", ctypes.c_float),
        ("top_k", ctypes.c_int32), ("num_levels", ctypes.c_int32), ("strides", ctypes.c_int32 * 4),
        ("cell_px", ctypes.c_int32), ("sigma_cells", ctypes.c_float), ("truncate_sigmas", ctypes.c_float),
    ]


BOX_DTYPE = np.dtype([("x1", "<f4"), ("y1", "<f4"), ("x2", "<f4"), ("y2", "<f4"), ("score", "<f4"), ("cand_index", "<i4")])


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no fast-math): every fp32 op separately rounded."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
                               "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.oracle_half_to_float.restype = ctypes.c_float
        L.oracle_half_to_float.argtypes = [ctypes.c_uint16]
        L.oracle_logit_threshold.restype = ctypes.c_float
        L.oracle_logit_threshold.argtypes = [ctypes.c_float]
        L.oracle_iou.restype = ctypes.c_float
        L.oracle_iou.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_fold.restype = ctypes.c_int32
        L.oracle_fold.argtypes = [ctypes.c_int32, ctypes.c_int32]
        L.oracle_taps.restype = ctypes.c_int32
        L.oracle_taps.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_void_p]
        L.oracle_decode_candidate.restype = None
        L.oracle_decode_candidate.argtypes = [ctypes.POINTER(OracleParams), ctypes.c_int32, ctypes.c_int32, ctypes.c_int64,
                                              ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_nms_sorted.restype = ctypes.c_int32
        L.oracle_nms_sorted.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_float, ctypes.c_void_p]
        L.oracle_density.restype = ctypes.c_int32
        L.oracle_density.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                     ctypes.c_float, ctypes.c_float, ctypes.c_void_p]
        L.oracle_run.restype = ctypes.c_int32
        L.oracle_run.argtypes = [ctypes.POINTER(OracleParams), ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p,
                                 ctypes.c_void_p] + [ctypes.c_void_p] * 6
        _lib = L
    return _lib


def make_params(params: dict) -> OracleParams:
    p = OracleParams()
    p.dtype = 1 if params["dtype"] == "fp16" else 0
    p.conf_thresh = params["conf_thresh"]
    p.iou_thresh = params["iou_thresh"]
    p.top_k = params["top_k"]
    strides = params.get("strides", [8, 16, 32])
    p.num_levels = len(strides)
    for i, s in enumerate(strides):
        p.strides[i] = s
    p.cell_px = params.get("cell_px", 8)
    p.sigma_cells = params["sigma_cells"]
    p.truncate_sigmas = params.get("truncate_sigmas", 3.0)
    return p


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def logit_threshold(conf: float) -> float:
    return float(lib().oracle_logit_threshold(conf))


def half_to_float(bits: int) -> float:
    return float(lib().oracle_half_to_float(bits))


def iou(a, b) -> float:
    a = np.ascontiguousarray(a, dtype=np.float32)
    b = np.ascontiguousarray(b, dtype=np.float32)
    return float(lib().oracle_iou(_ptr(a), _ptr(b)))


def fold(i: int, n: int) -> int:
    return int(lib().oracle_fold(i, n))


def taps(sigma: float, truncate: float = 3.0):
    R = lib().oracle_taps(sigma, truncate, None)
    w = np.zeros(2 * R + 1, dtype=np.float64)
    lib().oracle_taps(sigma, truncate, _ptr(w))
    return int(R), w


def decode_candidate(params: dict, W: int, H: int, j: int, ltrb):
    p = make_params(params)
    v = np.ascontiguousarray(ltrb, dtype=np.float32)
    out = np.zeros(4, dtype=np.float32)
    loc = np.zeros(3, dtype=np.int32)
    lib().oracle_decode_candidate(ctypes.byref(p), W, H, j, _ptr(v), _ptr(out), _ptr(loc))
    return out, tuple(int(x) for x in loc)


def nms_sorted(boxes, thr: float):
    b = np.ascontiguousarray(boxes, dtype=np.float32).reshape(-1, 4)
    keep = np.zeros(max(len(b), 1), dtype=np.int32)
    n = lib().oracle_nms_sorted(_ptr(b), len(b), thr, _ptr(keep))
    return keep[:n].copy()


def density(boxes, W: int, H: int, cell: int, sigma: float, truncate: float = 3.0):
    b = np.ascontiguousarray(boxes, dtype=np.float32).reshape(-1, 4)
    out = np.zeros((H // cell, W // cell), dtype=np.float32)
    n_in = lib().oracle_density(_ptr(b), len(b), W, H, cell, sigma, truncate, _ptr(out))
    return out, int(n_in)


class Result:
    __slots__ = ("boxes", "counts", "density", "density_offsets", "sorted_idx", "sorted_counts", "survivor_counts")


def run(params: dict, raw: np.ndarray, N_per_frame, frame_dims) -> Result:
    """Whole path on host arrays.  raw: [sum N, 5] float16/float32."""
    p = make_params(params)
    raw = np.ascontiguousarray(raw)
    assert raw.dtype == (np.float16 if p.dtype == 1 else np.float32)
    N = np.ascontiguousarray(N_per_frame, dtype=np.int32)
    dims = np.ascontiguousarray(frame_dims, dtype=np.int32).reshape(-1, 2)
    B = len(N)
    assert raw.shape[0] == int(N.sum())
    K = p.top_k
    cells = (dims[:, 0] // p.cell_px).astype(np.int64) * (dims[:, 1] // p.cell_px)
    r = Result()
    r.boxes = np.zeros((B, K), dtype=BOX_DTYPE)
    r.counts = np.zeros(B, dtype=np.int32)
    r.density = np.zeros(int(cells.sum()), dtype=np.float32)
    r.density_offsets = np.concatenate([[0], np.cumsum(cells)]).astype(np.int64)
    r.sorted_idx = np.full((B, K), -1, dtype=np.int32)
    r.sorted_counts = np.zeros(B, dtype=np.int32)
    r.survivor_counts = np.zeros(B, dtype=np.int32)
    if B == 0:
        return r
    rc = lib().oracle_run(ctypes.byref(p), _ptr(raw), B, _ptr(N), _ptr(dims), _ptr(r.boxes), _ptr(r.counts),
                          _ptr(r.density), _ptr(r.sorted_idx), _ptr(r.sorted_counts), _ptr(r.survivor_counts))
    if rc != 0:
        raise RuntimeError(f"oracle_run failed: {rc}")
    return r
