"""paper_2512_07009_b200 — Python binding of libffpp (include/ffpp.h).

Argument marshalling only: every step of the path (threshold/compaction, top-K select + decode + spatial
binning, NMS suppression pairs, greedy resolve + output gather, density) runs in the hand-written sm_100a
kernels of ``csrc/``.  PyTorch supplies device
memory and streams, nothing else.  There is no CPU fallback: if the CUDA library is missing or no
sm_100 device is present, construction raises.

    from paper_2512_07009_b200 import FFPP
    pp = FFPP(params, max_frames=B, max_total_candidates=N_total, max_frame_w=W, max_frame_h=H)
    out = pp.run(raw_cuda_tensor, N_per_frame, frame_dims)          # ffpp_run: device buffers, async
    out = pp.run_host(raw_numpy, N_per_frame, frame_dims)           # ffpp_run_host: host buffers, synchronous
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libffpp.so")
_SOURCES = ["ffpp.cu", "ffpp_kernels.cuh", "ffpp_common.cuh", "ffpp_next.cuh"]
_INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]

FFPP_OK, FFPP_EINVAL, FFPP_ECAPACITY, FFPP_ECUDA, FFPP_ENOMEM = 0, -1, -2, -3, -4
NUM_STAGES = 6
STAGE_NAMES = ["a0_schedule", "a1_threshold_compact", "a2_select_decode_bin", "a3_nms_pairs", "a4_nms_resolve_emit", "a5a6_density"]

STAGE_KERNELS = {"a0_schedule": "host scheduler + k0_clear", "a1_threshold_compact": "k1_threshold_compact",
                 "a2_select_decode_bin": "k2_select_bin", "a3_nms_pairs": "k3_nms_edges",
                 "a4_nms_resolve_emit": "k4_resolve_order + k4e_emit", "a5a6_density": "k5_density"}
# kernel launches of one ffpp_run (k0_clear, k1, k2, k3, k4, k4e, k5); no memset; on first sight of a
# batch geometry, one descriptor upload
LAUNCHES_PER_RUN = 7

# fp32 instructions per IoU pair of the all-pairs bitmask method (4 min/max, 2 sub, 2 clamp, 1 mul, area
# add/sub, divide-or-multiply + compare = 12-16; 15 taken).  bench.py divides the fp32 lane rate by this to get the
# pairs/s ceiling of the all-pairs method (DESIGN.md §6 a3).
NMS_ALU_OPS_PER_PAIR = 15

BOX_DTYPE = np.dtype([("x1", "<f4"), ("y1", "<f4"), ("x2", "<f4"), ("y2", "<f4"), ("score", "<f4"), ("cand_index", "<i4")])

EXPORTS = ["ffpp_create", "ffpp_run", "ffpp_run_host", "ffpp_destroy", "ffpp_last_error", "ffpp_get_info",
           "ffpp_set_stage_timing", "ffpp_get_stage_ms"]
DEBUG_EXPORTS = ["ffpp_debug_read", "ffpp_debug_count_work", "ffpp_debug_stream_read"]     # include/ffpp_debug.h
NEXT_EXPORTS = ["ffpp_heatmap_stats", "ffpp_density_exact", "ffpp_mask_components", "ffpp_preprocess"]   # include/ffpp_next.h
NOALLOC_EXPORTS = ["ffpp_heatmap_entropy_noalloc"]                                                       # include/ffpp_noalloc.h
NOALLOC_MAX_BLOCKS = 16384          # FFPP_NOALLOC_MAX_BLOCKS: B * ceil(gw*gh/2048) per call

REGION_DTYPE = np.dtype([("label", "<i4"), ("area", "<i4"), ("x0", "<i4"), ("y0", "<i4"), ("x1", "<i4"), ("y1", "<i4"),
                         ("mass", "<f4"), ("reserved_", "<i4")])


class FFPPParams(ctypes.Structure):
    _fields_ = [
        ("dtype", ctypes.c_int32), ("conf_thresh", ctypes.c_float), ("iou_thresh", ctypes.c_float),
        ("top_k", ctypes.c_int32), ("num_levels", ctypes.c_int32), ("strides", ctypes.c_int32 * 4),
        ("cell_px", ctypes.c_int32), ("sigma_cells", ctypes.c_float), ("truncate_sigmas", ctypes.c_float),
        ("max_frames", ctypes.c_int32), ("max_total_candidates", ctypes.c_int64),
        ("max_frame_w", ctypes.c_int32), ("max_frame_h", ctypes.c_int32),
        ("max_total_cells", ctypes.c_int64), ("nms_workspace_bytes", ctypes.c_int64),
        ("nms_edges_per_box", ctypes.c_int32), ("reserved_", ctypes.c_int32),
    ]


class FFPPInfo(ctypes.Structure):
    _fields_ = [
        ("logit_threshold", ctypes.c_float), ("radius", ctypes.c_int32), ("taps", ctypes.c_float * 65),
        ("key_bits", ctypes.c_int32), ("workspace_bytes", ctypes.c_int64), ("sm_count", ctypes.c_int32),
    ]


class FFPPError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libffpp error {code}: {msg}")
        self.code = code


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ffpp.cu for sm_100a into libffpp.so next to this file (nvcc cross-compiles without a GPU)."""
    srcs = [os.path.join(_CSRC, s) for s in _SOURCES] + [os.path.join(_INCLUDE, "ffpp.h"), os.path.join(_INCLUDE, "ffpp_debug.h"), os.path.join(_INCLUDE, "ffpp_next.h"),
                                                     os.path.join(_INCLUDE, "ffpp_noalloc.h")]
    stale = not os.path.exists(_LIB) or any(os.path.getmtime(s) > os.path.getmtime(_LIB) for s in srcs)
    if force or stale:
        cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", _LIB, os.path.join(_CSRC, "ffpp.cu")]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libffpp.so (building it first if sources are newer); raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = build()
        L = ctypes.CDLL(path)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        L.ffpp_create.restype = ctypes.c_int
        L.ffpp_create.argtypes = [ctypes.POINTER(FFPPParams), ctypes.POINTER(vp)]
        for name in ("ffpp_run", "ffpp_run_host"):
            fn = getattr(L, name)
            fn.restype = ctypes.c_int
            fn.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, vp]
        L.ffpp_destroy.restype = ctypes.c_int
        L.ffpp_destroy.argtypes = [vp]
        L.ffpp_last_error.restype = ctypes.c_char_p
        L.ffpp_last_error.argtypes = [vp]
        L.ffpp_get_info.restype = ctypes.c_int
        L.ffpp_get_info.argtypes = [vp, ctypes.POINTER(FFPPInfo)]
        L.ffpp_set_stage_timing.restype = ctypes.c_int
        L.ffpp_set_stage_timing.argtypes = [vp, i32]
        L.ffpp_get_stage_ms.restype = ctypes.c_int
        L.ffpp_get_stage_ms.argtypes = [vp, vp]
        L.ffpp_debug_read.restype = ctypes.c_int
        L.ffpp_debug_read.argtypes = [vp, i32, vp, i64]
        L.ffpp_debug_count_work.restype = ctypes.c_int
        L.ffpp_debug_count_work.argtypes = [vp, i32]
        L.ffpp_debug_stream_read.restype = ctypes.c_int
        L.ffpp_debug_stream_read.argtypes = [vp, vp, i64, vp]
        f32 = ctypes.c_float
        L.ffpp_heatmap_stats.restype = ctypes.c_int
        L.ffpp_heatmap_stats.argtypes = [vp, vp, i32, vp, f32, i32, i32, vp, vp, vp, vp, vp, vp]
        L.ffpp_density_exact.restype = ctypes.c_int
        L.ffpp_density_exact.argtypes = [vp, vp, vp, i32, vp, vp, vp]
        L.ffpp_mask_components.restype = ctypes.c_int
        L.ffpp_mask_components.argtypes = [vp, vp, i32, i32, i32, i32, f32, i32, i32, i32, vp, vp, vp, vp]
        L.ffpp_preprocess.restype = ctypes.c_int
        L.ffpp_preprocess.argtypes = [vp, i32, i32, i32, i32, i32, vp, vp, i32, vp, vp]
        L.ffpp_heatmap_entropy_noalloc.restype = ctypes.c_int
        L.ffpp_heatmap_entropy_noalloc.argtypes = [vp, i32, i32, i32, vp, vp, vp]
        _lib = L
    return _lib


def make_params(params: dict, *, max_frames: int, max_total_candidates: int, max_frame_w: int, max_frame_h: int,
                max_total_cells: int = 0, nms_workspace_bytes: int = 0, nms_edges_per_box: int = 0) -> FFPPParams:
    p = FFPPParams()
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
    p.max_frames = max_frames
    p.max_total_candidates = max_total_candidates
    p.max_frame_w, p.max_frame_h = max_frame_w, max_frame_h
    p.max_total_cells = max_total_cells
    p.nms_workspace_bytes = nms_workspace_bytes
    p.nms_edges_per_box = nms_edges_per_box
    return p


class Output:
    """Views of one run's results.  `boxes` [B, top_k, 6] float32 (last column = cand_index bits), `counts` [B]
    int32, `density` flat float32 with `density_offsets` [B+1]."""
    __slots__ = ("boxes", "counts", "density", "density_offsets")

    def boxes_numpy(self) -> np.ndarray:
        b = self.boxes.cpu().numpy() if hasattr(self.boxes, "cpu") else self.boxes
        return np.ascontiguousarray(b).view(BOX_DTYPE).reshape(b.shape[0], b.shape[1])

    def counts_numpy(self) -> np.ndarray:
        return self.counts.cpu().numpy() if hasattr(self.counts, "cpu") else self.counts

    def density_numpy(self) -> np.ndarray:
        return self.density.cpu().numpy() if hasattr(self.density, "cpu") else self.density


class FFPP:
    """One libffpp handle (ffpp_create / ffpp_destroy) on the current CUDA device."""

    def __init__(self, params: dict, *, max_frames: int, max_total_candidates: int, max_frame_w: int, max_frame_h: int,
                 max_total_cells: int = 0, nms_workspace_bytes: int = 0, nms_edges_per_box: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2512_07009_b200 needs a CUDA sm_100 device; there is no CPU fallback")
        torch.cuda.init()
        self._torch = torch
        self._lib = load_library()
        self.params = dict(params)
        self.top_k = int(params["top_k"])
        self.cell_px = int(params.get("cell_px", 8))
        self._np_dtype = np.float16 if params["dtype"] == "fp16" else np.float32
        self._torch_dtype = torch.float16 if params["dtype"] == "fp16" else torch.float32
        self._p = make_params(params, max_frames=max_frames, max_total_candidates=max_total_candidates,
                              max_frame_w=max_frame_w, max_frame_h=max_frame_h, max_total_cells=max_total_cells,
                              nms_workspace_bytes=nms_workspace_bytes, nms_edges_per_box=nms_edges_per_box)
        self._h = ctypes.c_void_p()
        rc = self._lib.ffpp_create(ctypes.byref(self._p), ctypes.byref(self._h))
        if rc != FFPP_OK:
            self._h = ctypes.c_void_p()
            raise FFPPError(rc, self._lib.ffpp_last_error(None).decode())

    @classmethod
    def for_workload(cls, w, **kw) -> "FFPP":
        """Handle sized exactly for a flockgen.Workload-like object (params, N_per_frame, frame_dims)."""
        dims = np.asarray(w.frame_dims).reshape(-1, 2)
        return cls(w.params, max_frames=max(1, len(w.N_per_frame)), max_total_candidates=max(1, int(np.sum(w.N_per_frame))),
                   max_frame_w=int(dims[:, 0].max()) if len(dims) else 64, max_frame_h=int(dims[:, 1].max()) if len(dims) else 64,
                   **kw)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.ffpp_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc != FFPP_OK:
            raise FFPPError(rc, self._lib.ffpp_last_error(self._h).decode())

    def info(self) -> FFPPInfo:
        out = FFPPInfo()
        self._check(self._lib.ffpp_get_info(self._h, ctypes.byref(out)))
        return out

    @staticmethod
    def _host_i32(a, shape):
        return np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(shape))

    def density_offsets(self, frame_dims) -> np.ndarray:
        d = np.asarray(frame_dims, dtype=np.int64).reshape(-1, 2)
        return np.concatenate([[0], np.cumsum((d[:, 0] // self.cell_px) * (d[:, 1] // self.cell_px))]).astype(np.int64)

    def alloc_outputs(self, B: int, frame_dims) -> Output:
        torch = self._torch
        out = Output()
        out.density_offsets = self.density_offsets(frame_dims)
        out.boxes = torch.empty((B, self.top_k, 6), dtype=torch.float32, device="cuda")
        out.counts = torch.empty((B,), dtype=torch.int32, device="cuda")
        out.density = torch.empty((int(out.density_offsets[-1]),), dtype=torch.float32, device="cuda")
        return out

    def run(self, raw, N_per_frame, frame_dims, out: Output | None = None, stream=None) -> Output:
        """ffpp_run: `raw` is a CUDA tensor [sum N, 5] of the handle's dtype.  Asynchronous on `stream`
        (default: torch's current stream)."""
        torch = self._torch
        N = self._host_i32(N_per_frame, (-1,))
        dims = self._host_i32(frame_dims, (-1, 2))
        B = int(N.shape[0])
        if out is None:
            out = self.alloc_outputs(B, dims)
        if B:
            assert raw.is_cuda and raw.dtype == self._torch_dtype and raw.is_contiguous()
        st = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.ffpp_run(self._h, raw.data_ptr() if B else None, B, N.ctypes.data, dims.ctypes.data,
                                       st.cuda_stream, out.boxes.data_ptr(), out.counts.data_ptr(), out.density.data_ptr()))
        return out

    def run_raw_pointers(self, raw_ptr, B, N_ptr, dims_ptr, stream_ptr, boxes_ptr, counts_ptr, density_ptr) -> int:
        """Direct ffpp_run with caller-supplied addresses; returns the status code (for ABI misuse tests)."""
        return int(self._lib.ffpp_run(self._h, raw_ptr, B, N_ptr, dims_ptr, stream_ptr, boxes_ptr, counts_ptr, density_ptr))

    def last_error(self) -> str:
        return self._lib.ffpp_last_error(self._h).decode()

    def run_host(self, raw: np.ndarray, N_per_frame, frame_dims, out: Output | None = None, stream=None) -> Output:
        """ffpp_run_host: numpy (or pinned torch CPU) buffers in and out; synchronises before returning."""
        torch = self._torch
        N = self._host_i32(N_per_frame, (-1,))
        dims = self._host_i32(frame_dims, (-1, 2))
        B = int(N.shape[0])
        if out is None:
            out = Output()
            out.density_offsets = self.density_offsets(dims)
            out.boxes = np.zeros((B, self.top_k, 6), dtype=np.float32)
            out.counts = np.zeros((B,), dtype=np.int32)
            out.density = np.zeros((int(out.density_offsets[-1]),), dtype=np.float32)

        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data

        st = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.ffpp_run_host(self._h, ptr(raw) if B else None, B, N.ctypes.data, dims.ctypes.data,
                                            st.cuda_stream, ptr(out.boxes), ptr(out.counts), ptr(out.density)))
        return out

    # ---- measurement / debug helpers (thin wrappers of the C ABI) ----
    def set_stage_timing(self, enable: bool):
        self._check(self._lib.ffpp_set_stage_timing(self._h, 1 if enable else 0))

    def stage_ms(self) -> np.ndarray:
        ms = np.zeros(NUM_STAGES, dtype=np.float32)
        self._check(self._lib.ffpp_get_stage_ms(self._h, ms.ctypes.data))
        return ms

    def stream_read(self, dev_tensor, stream=None):
        """ffpp_debug_stream_read: enqueue a plain read of a device tensor (calibration of the a1 roofline)."""
        st = stream if stream is not None else self._torch.cuda.current_stream()
        self._check(self._lib.ffpp_debug_stream_read(self._h, dev_tensor.data_ptr(), dev_tensor.numel() * dev_tensor.element_size(),
                                                     st.cuda_stream))

    def count_work(self, enable: bool):
        """ffpp_debug_count_work: the next runs launch the counting instantiation of the a3 kernel."""
        self._check(self._lib.ffpp_debug_count_work(self._h, 1 if enable else 0))

    def debug_read(self, what: int, B: int) -> np.ndarray:
        K = self.top_k
        if what in (0, 1, 5):
            a = np.zeros(B, dtype=np.int32)
        elif what == 4:
            a = np.zeros(4, dtype=np.int64)
        elif what == 2:
            a = np.zeros((B, K), dtype=np.int32)
        else:
            a = np.zeros((B, K, 4), dtype=np.float32)
        self._check(self._lib.ffpp_debug_read(self._h, what, a.ctypes.data, a.nbytes))
        return a


    # ---- SURVEY §8(f) f1-f3 (include/ffpp_next.h): argument marshalling only ----
    def heatmap_stats(self, density, frame_dims, threshold: float, *, connectivity: int = 4, max_regions: int = 1024, stream=None):
        """ffpp_heatmap_stats.  density: CUDA float32 tensor in ffpp_run's out_density layout.  Returns a dict of CUDA
        tensors: entropy [B] f64, degree [B] f64, labels [cells] i32, regions [B, max_regions, 8] i32 (view with
        REGION_DTYPE), region_counts [B] i32."""
        torch = self._torch
        dims = self._host_i32(frame_dims, (-1, 2))
        B = int(dims.shape[0])
        assert density.is_cuda and density.dtype == torch.float32 and density.is_contiguous()
        res = {"entropy": torch.empty(B, dtype=torch.float64, device="cuda"), "degree": torch.empty(B, dtype=torch.float64, device="cuda"),
               "labels": torch.empty(density.numel(), dtype=torch.int32, device="cuda"),
               "regions": torch.zeros((B, max_regions, 8), dtype=torch.int32, device="cuda"),
               "region_counts": torch.empty(B, dtype=torch.int32, device="cuda")}
        st = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.ffpp_heatmap_stats(self._h, density.data_ptr(), B, dims.ctypes.data, threshold, connectivity, max_regions,
                                                 st.cuda_stream, res["entropy"].data_ptr(), res["degree"].data_ptr(), res["labels"].data_ptr(),
                                                 res["regions"].data_ptr(), res["region_counts"].data_ptr()))
        return res

    def density_exact(self, out: Output, frame_dims, stream=None):
        """ffpp_density_exact on the kept boxes of a finished run; returns a CUDA float32 tensor in the out_density layout."""
        torch = self._torch
        dims = self._host_i32(frame_dims, (-1, 2))
        B = int(dims.shape[0])
        dens = torch.empty(int(self.density_offsets(dims)[-1]), dtype=torch.float32, device="cuda")
        st = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.ffpp_density_exact(self._h, out.boxes.data_ptr(), out.counts.data_ptr(), B, dims.ctypes.data, st.cuda_stream,
                                                 dens.data_ptr()))
        return dens

    def mask_components(self, mask, threshold: float, *, connectivity: int = 8, min_area: int = 1, max_components: int = 4096, stream=None):
        """ffpp_mask_components.  mask: CUDA tensor [B, H, W] float16/float32.  Returns dict: labels [B, H, W] i32,
        components [B, max_components, 8] i32 (REGION_DTYPE; mass = mean probability), counts [B] i32."""
        torch = self._torch
        assert mask.is_cuda and mask.is_contiguous() and mask.dim() == 3 and mask.dtype in (torch.float16, torch.float32)
        B, H, W = (int(v) for v in mask.shape)
        res = {"labels": torch.empty((B, H, W), dtype=torch.int32, device="cuda"),
               "components": torch.zeros((B, max_components, 8), dtype=torch.int32, device="cuda"),
               "counts": torch.empty(B, dtype=torch.int32, device="cuda")}
        st = stream if stream is not None else torch.cuda.current_stream()
        self._check(self._lib.ffpp_mask_components(self._h, mask.data_ptr(), 1 if mask.dtype == torch.float16 else 0, B, W, H, threshold,
                                                   connectivity, min_area, max_components, st.cuda_stream, res["labels"].data_ptr(),
                                                   res["components"].data_ptr(), res["counts"].data_ptr()))
        return res


def regions_numpy(t) -> np.ndarray:
    """[B, max, 8] int32 CUDA/CPU tensor of ffpp_region records -> numpy structured array [B, max]."""
    a = t.cpu().numpy() if hasattr(t, "cpu") else np.asarray(t)
    return np.ascontiguousarray(a).view(REGION_DTYPE).reshape(a.shape[0], a.shape[1])


def preprocess(src, Hd: int, Wd: int, mean, std, *, out_dtype="fp16", stream=None):
    """ffpp_preprocess.  src: CUDA uint8 tensor [B, Hs, Ws, 3] -> CUDA tensor [B, 3, Hd, Wd] float16/float32."""
    import torch
    lib = load_library()
    assert src.is_cuda and src.dtype == torch.uint8 and src.is_contiguous() and src.dim() == 4 and src.shape[3] == 3
    B, Hs, Ws, _ = (int(v) for v in src.shape)
    dst = torch.empty((B, 3, Hd, Wd), dtype=torch.float16 if out_dtype == "fp16" else torch.float32, device="cuda")
    m = np.ascontiguousarray(mean, dtype=np.float32)
    s = np.ascontiguousarray(std, dtype=np.float32)
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib.ffpp_preprocess(src.data_ptr(), B, Hs, Ws, Hd, Wd, m.ctypes.data, s.ctypes.data, 1 if out_dtype == "fp16" else 0, st.cuda_stream,
                             dst.data_ptr())
    if rc != FFPP_OK:
        raise FFPPError(rc, "ffpp_preprocess")
    return dst


def heatmap_entropy_noalloc(density, gw: int, gh: int, out_entropy, out_degree, stream=None) -> None:
    """ffpp_heatmap_entropy_noalloc (include/ffpp_noalloc.h): density is a CUDA float32 tensor [B, gh, gw]; the two outputs
    are caller-allocated CUDA float64 tensors [B].  The library allocates nothing (static 256 KiB device scratch)."""
    import torch
    lib = load_library()
    assert density.is_cuda and density.dtype == torch.float32 and density.is_contiguous()
    B = int(density.numel() // (gw * gh)) if gw > 0 and gh > 0 else 0
    assert out_entropy.is_cuda and out_degree.is_cuda and out_entropy.dtype == torch.float64 and out_degree.dtype == torch.float64
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = lib.ffpp_heatmap_entropy_noalloc(density.data_ptr(), B, gw, gh, st.cuda_stream, out_entropy.data_ptr(), out_degree.data_ptr())
    if rc != FFPP_OK:
        raise FFPPError(rc, lib.ffpp_last_error(None).decode())
