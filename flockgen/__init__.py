"""flockgen — seeded synthetic flock workloads (input generator; no post-processing code).

Stands in for the paper's private farm videos and detector outputs (§4), with
the shapes / distributions of BASELINE.json ``configs[0..4]``.  Used as
*input* by the oracle tests, the GPU parity tests and ``bench.py``.  It imports neither
``oracle`` nor the CUDA package.

    cfg = flockgen.make_config(2, seed_offset=0)
    cfg.raw            # numpy [sum N_f, 5] float16/float32 (l,t,r,b in stride units, score logit)
    cfg.N_per_frame    # int32 [B]
    cfg.frame_dims     # int32 [B,2] = (W,H)
    cfg.params         # dict: dtype, conf_thresh, iou_thresh, top_k, strides, cell_px, sigma_cells, truncate_sigmas
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "flockgen.cpp")
_LIB = os.path.join(_HERE, "libflockgen.so")

STRIDES = (8, 16, 32)


class _FrameSpec(ctypes.Structure):
    _fields_ = [
        ("W", ctypes.c_int32), ("H", ctypes.c_int32),
        ("lambda_lo", ctypes.c_double), ("lambda_hi", ctypes.c_double), ("lambda_cap", ctypes.c_double),
        ("box_median", ctypes.c_double), ("box_sigma", ctypes.c_double),
        ("layout", ctypes.c_int32), ("n_components", ctypes.c_int32),
        ("comp_sigma", ctypes.c_double), ("frac", ctypes.c_double),
        ("bg_beta_a", ctypes.c_int32), ("bg_beta_b", ctypes.c_int32),
    ]


class _Params(ctypes.Structure):
    _fields_ = [
        ("dtype", ctypes.c_int32), ("num_levels", ctypes.c_int32), ("strides", ctypes.c_int32 * 4),
        ("conf_thresh", ctypes.c_double), ("iou_thresh", ctypes.c_double), ("top_k", ctypes.c_int32),
        ("jitter_px", ctypes.c_double), ("iou_margin", ctypes.c_double), ("threads", ctypes.c_int32),
    ]


class _Stats(ctypes.Structure):
    _fields_ = [("birds", ctypes.c_int64), ("redraws", ctypes.c_int64), ("evicted", ctypes.c_int64)]


def build(force: bool = False) -> str:
    """Compile libflockgen.so in-tree (g++ only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.flockgen_generate.restype = ctypes.c_int
        lib.flockgen_generate.argtypes = [ctypes.POINTER(_Params), ctypes.c_int32, ctypes.POINTER(_FrameSpec),
                                          ctypes.c_uint64, ctypes.c_void_p, ctypes.POINTER(_Stats)]
        _lib = lib
    return _lib


def frame_candidates(W: int, H: int, strides=STRIDES) -> int:
    """N_f = sum_l W*H/s_l^2 (1280x720 -> 18900 per A21)."""
    return sum((W * H) // (s * s) for s in strides)


@dataclass
class Workload:
    name: str
    raw: np.ndarray
    N_per_frame: np.ndarray
    frame_dims: np.ndarray
    params: dict
    seed: int
    stats: dict = field(default_factory=dict)

    @property
    def B(self) -> int:
        return int(self.N_per_frame.shape[0])

    @property
    def total_candidates(self) -> int:
        return int(self.N_per_frame.sum())

    def grid_cells(self) -> np.ndarray:
        c = self.params["cell_px"]
        return (self.frame_dims[:, 0] // c) * (self.frame_dims[:, 1] // c)


def _spec(W, H, lam, median, layout=0, ncomp=3, comp_sigma=60.0, frac=0.2, bg=(1, 20), lam_hi=0.0, lam_cap=0.0):
    return dict(W=W, H=H, lambda_lo=float(lam), lambda_hi=float(lam_hi), lambda_cap=float(lam_cap),
                box_median=float(median), box_sigma=0.25, layout=layout, n_components=ncomp,
                comp_sigma=float(comp_sigma), frac=float(frac), bg_beta_a=bg[0], bg_beta_b=bg[1])


def generate(name: str, specs: list[dict], *, dtype: str, conf: float, iou: float, top_k: int, sigma_cells: float,
             seed: int, cell_px: int = 8, truncate_sigmas: float = 3.0, threads: int = 0,
             iou_margin: float = 1e-5) -> Workload:
    """Generate one batch from explicit per-frame specs (see ``_spec``)."""
    lib = _load()
    B = len(specs)
    pa = _Params()
    pa.dtype = 1 if dtype == "fp16" else 0
    pa.num_levels = len(STRIDES)
    for i, s in enumerate(STRIDES):
        pa.strides[i] = s
    pa.conf_thresh, pa.iou_thresh, pa.top_k = conf, iou, top_k
    pa.jitter_px, pa.iou_margin, pa.threads = 1.5, iou_margin, threads
    arr = (_FrameSpec * max(B, 1))()
    for i, s in enumerate(specs):
        for k, v in s.items():
            setattr(arr[i], k, v)
    N = np.array([frame_candidates(s["W"], s["H"]) for s in specs], dtype=np.int32).reshape(B)
    dims = np.array([[s["W"], s["H"]] for s in specs], dtype=np.int32).reshape(B, 2)
    raw = np.zeros((int(N.sum()), 5), dtype=np.float16 if dtype == "fp16" else np.float32)
    st = _Stats()
    rc = lib.flockgen_generate(ctypes.byref(pa), B, arr, ctypes.c_uint64(seed & (2**64 - 1)),
                               raw.ctypes.data_as(ctypes.c_void_p), ctypes.byref(st))
    if rc != 0:
        raise RuntimeError(f"flockgen_generate failed: {rc}")
    params = dict(dtype=dtype, conf_thresh=conf, iou_thresh=iou, top_k=top_k, strides=list(STRIDES),
                  cell_px=cell_px, sigma_cells=sigma_cells, truncate_sigmas=truncate_sigmas)
    return Workload(name=name, raw=raw, N_per_frame=N, frame_dims=dims, params=params, seed=seed,
                    stats=dict(birds=st.birds, redraws=st.redraws, evicted=st.evicted))


def config_seed(c: int) -> int:
    """seed_c of SURVEY §8(d): 0x251207009 ^ (c * golden-ratio constant), 64-bit."""
    return (0x251207009 ^ ((c * 0x9E3779B97F4A7C15) & (2**64 - 1))) & (2**64 - 1)


def config_specs(c: int, B: int | None = None):
    """Per-frame specs + method parameters of BASELINE.json configs[c-1] (c = 1..5).

    ``B`` overrides the batch size (same per-frame recipe) for reduced parity cases."""
    if c == 1:
        specs = [_spec(640, 640, 150, 40)] * (B or 1)
        kw = dict(dtype="fp32", conf=0.25, iou=0.45, top_k=3000, sigma_cells=2.0)
    elif c == 2:
        specs = [_spec(640, 640, 300, 40)] * (B or 16)
        kw = dict(dtype="fp16", conf=0.25, iou=0.45, top_k=3000, sigma_cells=2.0)
    elif c == 3:  # mixture concentrated near 4 feeder/drinker sites
        specs = [_spec(1280, 1280, 800, 30, ncomp=4, comp_sigma=100.0)] * (B or 32)
        kw = dict(dtype="fp16", conf=0.2, iou=0.5, top_k=8000, sigma_cells=2.5)
    elif c == 4:  # dense flock: uniform + 30 % clustered neighbours
        specs = [_spec(1920, 1088, 2000, 24, layout=1, frac=0.3)] * (B or 64)
        kw = dict(dtype="fp16", conf=0.15, iou=0.45, top_k=12000, sigma_cells=3.0)
    elif c == 5:  # ragged multi-zone batch, interleaved resolutions, every 4th of each res is clutter
        res = [(640, 640, 400.0), (1280, 1280, 0.0), (1920, 1088, 0.0), (1280, 720, 1200.0)]
        specs = []
        for f in range(B or 256):
            W, H, cap = res[f % 4]
            clutter = (f // 4) % 4 == 3
            specs.append(_spec(W, H, 100, 30, comp_sigma=60.0 * W / 640.0, lam_hi=2500, lam_cap=cap,
                               bg=(2, 5) if clutter else (1, 20)))
        kw = dict(dtype="fp16", conf=0.2, iou=0.5, top_k=12000, sigma_cells=2.5)
    else:
        raise ValueError("config must be 1..5")
    return specs, kw


def make_config(c: int, seed_offset: int = 0, B: int | None = None, threads: int = 0, iou_margin: float = 1e-5) -> Workload:
    """``iou_margin`` = 0 switches the IoU-margin rejection of SURVEY §8(d) step (7) off (parity cases only)."""
    specs, kw = config_specs(c, B)
    return generate(f"config{c}" + (f"_B{B}" if B else ""), specs, seed=config_seed(c) + seed_offset, threads=threads,
                    iou_margin=iou_margin, **kw)


# ---------------------------------------------------------------------------------------------------------------
# Inputs of the SURVEY §8(f) rows f3 / f4 (numpy only; stand-ins for the paper's UNeXt segmentation output and its
# 1080p / 720p farm video frames).  No method arithmetic: a probability mask is a sum of
# seeded blobs, an image is seeded smooth colour noise.
# ---------------------------------------------------------------------------------------------------------------
def make_mask_batch(B: int, W: int, H: int, *, birds: float = 300.0, seed: int = 0x2512_0700_9, dtype="fp16") -> np.ndarray:
    """[B, H, W] bird-segmentation probabilities in [0, 1]: Poisson(birds) elliptical blobs per frame (axes lognormal
    around 14 x 9 px, random orientation, peak 0.6-0.99, soft edge), some touching, plus low-level background noise."""
    rng = np.random.default_rng(seed)
    out = np.empty((B, H, W), dtype=np.float16 if dtype == "fp16" else np.float32)
    yy, xx = np.mgrid[0:H, 0:W].astype(np.float32)
    for b in range(B):
        m = rng.random((H, W), dtype=np.float32) * 0.25                 # background: well below any sane threshold ...
        speck = rng.random((H, W)) < 2e-4                               # ... plus isolated hot pixels (1-pixel components)
        m[speck] = 0.9
        nb = int(rng.poisson(birds))
        cx = rng.uniform(0, W, nb); cy = rng.uniform(0, H, nb)
        a = 14.0 * np.exp(rng.normal(0, 0.25, nb)); bb = 9.0 * np.exp(rng.normal(0, 0.25, nb))
        th = rng.uniform(0, np.pi, nb); pk = rng.uniform(0.6, 0.99, nb)
        for i in range(nb):
            x0, x1 = int(max(0, cx[i] - 3 * a[i])), int(min(W, cx[i] + 3 * a[i] + 1))
            y0, y1 = int(max(0, cy[i] - 3 * a[i])), int(min(H, cy[i] + 3 * a[i] + 1))
            if x0 >= x1 or y0 >= y1:
                continue
            dx = xx[y0:y1, x0:x1] - cx[i]; dy = yy[y0:y1, x0:x1] - cy[i]
            u = (dx * np.cos(th[i]) + dy * np.sin(th[i])) / a[i]
            v = (-dx * np.sin(th[i]) + dy * np.cos(th[i])) / bb[i]
            blob = pk[i] / (1.0 + np.exp(8.0 * (np.sqrt(u * u + v * v) - 1.0)))      # soft-edged ellipse
            np.maximum(m[y0:y1, x0:x1], blob.astype(np.float32), out=m[y0:y1, x0:x1])
        out[b] = m
    return out


def make_image_batch(B: int, W: int, H: int, *, seed: int = 0x2512_0700_9) -> np.ndarray:
    """[B, H, W, 3] uint8 frames: smooth colour gradients + blocks + pixel noise (every byte value occurs)."""
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W].astype(np.float32)
    out = np.empty((B, H, W, 3), dtype=np.uint8)
    for b in range(B):
        for c in range(3):
            fx, fy, ph = rng.uniform(0.002, 0.05), rng.uniform(0.002, 0.05), rng.uniform(0, 6.28)
            img = 127.5 + 100.0 * np.sin(fx * xx + fy * yy + ph) + rng.normal(0, 12.0, (H, W))
            out[b, :, :, c] = np.clip(img, 0, 255).astype(np.uint8)
        for _ in range(8):                                              # hard-edged blocks (sharp transitions)
            x0, y0 = int(rng.integers(0, W)), int(rng.integers(0, H))
            out[b, y0:y0 + int(rng.integers(4, 64)), x0:x0 + int(rng.integers(4, 64)), :] = rng.integers(0, 256, 3, dtype=np.uint8)
    return out
