"""ctypes binding of the CPU oracle (oracle/ffpp_oracle.cpp, oracle/ffpp_next_oracle.cpp) — TEST INFRASTRUCTURE.

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
_SRC_NEXT = os.path.join(_HERE, "ffpp_next_oracle.cpp")
_LIB_NEXT = os.path.join(_HERE, "libffpp_next_oracle.so")


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
    if force or not os.path.exists(_LIB_NEXT) or os.path.getmtime(_LIB_NEXT) < os.path.getmtime(_SRC_NEXT):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
                               "-o", _LIB_NEXT, _SRC_NEXT])
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


# ---------------------------------------------------------------------------------------------------------------
# SURVEY §8(f) f1-f4 (oracle/ffpp_next_oracle.cpp)
# ---------------------------------------------------------------------------------------------------------------
REGION_DTYPE = np.dtype([("label", "<i4"), ("area", "<i4"), ("x0", "<i4"), ("y0", "<i4"), ("x1", "<i4"), ("y1", "<i4"),
                         ("mass", "<f4"), ("reserved_", "<i4")])

_lib_next = None


def lib_next():
    global _lib_next
    if _lib_next is None:
        build()
        L = ctypes.CDLL(_LIB_NEXT)
        vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
        L.oracle_entropy.restype = ctypes.c_double
        L.oracle_entropy.argtypes = [vp, i64]
        L.oracle_clustering_degree.restype = ctypes.c_double
        L.oracle_clustering_degree.argtypes = [vp, i64]
        L.oracle_regions.restype = i32
        L.oracle_regions.argtypes = [vp, i32, i32, f32, i32, vp, vp, i32]
        L.oracle_density_exact.restype = i32
        L.oracle_density_exact.argtypes = [vp, i32, i32, i32, i32, f32, f32, vp]
        L.oracle_mask_components.restype = i32
        L.oracle_mask_components.argtypes = [vp, i32, i32, i32, f32, i32, i32, vp, vp, i32]
        L.oracle_preprocess.restype = None
        L.oracle_preprocess.argtypes = [vp, i32, i32, i32, i32, vp, vp, vp]
        _lib_next = L
    return _lib_next


def entropy(D) -> float:
    d = np.ascontiguousarray(D, dtype=np.float32).reshape(-1)
    return float(lib_next().oracle_entropy(_ptr(d), d.size))


def clustering_degree(D) -> float:
    d = np.ascontiguousarray(D, dtype=np.float32).reshape(-1)
    return float(lib_next().oracle_clustering_degree(_ptr(d), d.size))


def regions(D, thr: float, conn: int = 4, max_regions: int = 4096):
    """(labels [gh, gw] int32, table REGION_DTYPE[min(count, max_regions)], count)."""
    d = np.ascontiguousarray(D, dtype=np.float32)
    gh, gw = d.shape
    labels = np.zeros((gh, gw), dtype=np.int32)
    tab = np.zeros(max_regions, dtype=REGION_DTYPE)
    n = lib_next().oracle_regions(_ptr(d), gw, gh, thr, conn, _ptr(labels), _ptr(tab), max_regions)
    return labels, tab[:min(n, max_regions)].copy(), int(n)


def density_exact(boxes, W: int, H: int, cell: int, sigma: float, truncate: float = 3.0):
    b = np.ascontiguousarray(boxes, dtype=np.float32).reshape(-1, 4)
    out = np.zeros((H // cell, W // cell), dtype=np.float32)
    n_in = lib_next().oracle_density_exact(_ptr(b), len(b), W, H, cell, sigma, truncate, _ptr(out))
    return out, int(n_in)


def mask_components(mask, thr: float, conn: int = 8, min_area: int = 1, max_components: int = 8192):
    """mask [H, W] float16/float32 -> (labels [H, W] int32, table REGION_DTYPE (mass = mean probability), count)."""
    m = np.ascontiguousarray(mask)
    assert m.dtype in (np.float16, np.float32) and m.ndim == 2
    H, W = m.shape
    labels = np.zeros((H, W), dtype=np.int32)
    tab = np.zeros(max_components, dtype=REGION_DTYPE)
    n = lib_next().oracle_mask_components(_ptr(m), 1 if m.dtype == np.float16 else 0, W, H, thr, conn, min_area, _ptr(labels),
                                          _ptr(tab), max_components)
    return labels, tab[:min(n, max_components)].copy(), int(n)


def preprocess(img, Hd: int, Wd: int, mean, std) -> np.ndarray:
    """img [Hs, Ws, 3] uint8 -> [3, Hd, Wd] float64."""
    a = np.ascontiguousarray(img, dtype=np.uint8)
    Hs, Ws, _ = a.shape
    mean = np.ascontiguousarray(mean, dtype=np.float32)
    std = np.ascontiguousarray(std, dtype=np.float32)
    out = np.zeros((3, Hd, Wd), dtype=np.float64)
    lib_next().oracle_preprocess(_ptr(a), Hs, Ws, Hd, Wd, _ptr(mean), _ptr(std), _ptr(out))
    return out
