#!/usr/bin/env python
"""bench.py — throughput of the libffpp hot path on the synthetic flock workloads (BASELINE.json metric:
post-processed frames/s and candidates/s at 1 B200; % of roofline per stage).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

One "step" = one ffpp_run over one whole batch of the chosen config (all §8(a) rows a0-a6: seven kernel launches on
one stream, six of them programmatic dependents of their predecessor).  Default workload: config 5 (ragged 256-frame multi-zone batch, 6 639 360
candidates, 66.4 MB fp16), the largest single-GPU configuration and the only one that exercises the ragged
scheduler; the default single-GPU run also measures configs 1-4 briefly and carries them in `configs`.
Rank r of N generates its own batch (seed offset r): frames are independent, so N GPUs = N x the frames, no
data-path collective ("scaling": "weak").  `--gpus N` without a torchrun environment re-executes itself under
`python -m torch.distributed.run --nproc-per-node N`.

Timing: every timed step is bracketed by CUDA events on the launching stream.  Between steps L2 (126 MB) is left
COLD AND CLEAN: a 512 MB write evicts everything, then a 512 MB read (k0_stream_read) replaces the dirty lines of
that write with clean ones, so the step's first kernel does not compete with write-back traffic; both happen
outside the event pair.  The K step times are summed, the sum is max-reduced over ranks, and the timed loop sits
between barrier + torch.cuda.synchronize() on both sides.  `e2e` is the same metric through ffpp_run_host with
pinned HOST buffers (H2D of the raw head output and D2H of counts, density and kept boxes inside the timed
region).  `--impl reference` times the CPU oracle (oracle/) on a bounded sample; it is the only place besides
`cpu_baseline` where bench.py executes oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "post-processed frames/sec"
UNIT = "frames/s"

CONFIG_DESC = {
    1: "config1: B=1 640x640 fp32 [1,8400,5]",
    2: "config2: B=16 640x640 fp16 [16,8400,5]",
    3: "config3: B=32 1280x1280 fp16 [32,33600,5]",
    4: "config4: B=64 1920x1088 fp16 [64,42840,5]",
    5: "config5: ragged B=256 (64 each 640x640/1280x1280/1920x1088/1280x720, interleaved) fp16, 6639360 candidates",
}

# fp32 lane-instructions of the a3 method's own work (DESIGN.md §6 a3): every candidate pair of the cell
# windows gets the exact IoU, 15 fp32 instructions (4 min/max, 2 sub, 2 clamp, 1 mul, 2 area mul, 2 area sub, add, sub,
# multiply-or-divide + compare)
A3_OPS_PER_EXACT_IOU = 15
FP32_LANES_PER_SM = 128


def load_peaks():
    """Roofline denominators: driver-measured MEASURED_PEAKS.json, else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            p = json.load(fh)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def pair_count(n_sorted: np.ndarray) -> int:
    n = n_sorted.astype(np.int64)
    return int((n * (n - 1) // 2).sum())


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` outside a torchrun environment: start the N ranks ourselves (one process per GPU)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, cwd=ROOT)


# --------------------------------------------------------------------------------------------------------------
# reference arm: the oracle as it stands, on the host cores
# --------------------------------------------------------------------------------------------------------------
REF_SAMPLE_FRAMES = {1: 1, 2: 16, 3: 16, 4: 8, 5: 16}    # frames per reference "step" (bounded sample)
CPU_BASELINE_FRAMES = {1: 1, 2: 16, 3: 32, 4: 48, 5: 128}  # cpu_baseline sample of the default arm (~10-30 s)


def oracle_time(w, n_frames: int, reps: int = 1):
    """Seconds for the oracle over the first n_frames frames of workload w (single thread, as it stands)."""
    import oracle
    n_frames = min(n_frames, w.B)
    rows = int(w.N_per_frame[:n_frames].sum())
    raw = w.raw[:rows]
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.run(w.params, raw, w.N_per_frame[:n_frames], w.frame_dims[:n_frames])
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best, n_frames, rows


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import flockgen
    import oracle
    oracle.build()
    w = flockgen.make_config(args.config)
    nf = min(REF_SAMPLE_FRAMES[args.config], w.B)
    rows = int(w.N_per_frame[:nf].sum())
    for _ in range(args.warmup):
        oracle_time(w, nf)
    t = 0.0
    for _ in range(args.steps):
        t += oracle_time(w, nf)[0]
    fps = nf * args.steps / t
    sample = f"first {nf} of {w.B} frames of {w.name} per step ({rows} candidates), single thread"
    line = {
        "impl": "reference", "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": max(args.gpus, world), "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "input_dtype": w.params["dtype"], "data": "synthetic",
        "config": {"workload": CONFIG_DESC[args.config], "sample": sample},
        "candidates_per_s": rows * args.steps / t,
        "cpu_baseline": {"value": fps, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": fps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def reduce_over_ranks(total_ms: float, t_e2e: float, frames: float, cands: float, world: int, device):
    """Whole-job numbers of a weak-scaling run: times are the MAX over ranks, units are the SUM over ranks.
    No data-path collective exists (frames are independent); these two all-reduces are the only communication."""
    if world <= 1:
        return total_ms, t_e2e, frames, cands
    import torch
    import torch.distributed as dist
    t = torch.tensor([total_ms, t_e2e], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([frames, cands], dtype=torch.float64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(u[0]), float(u[1])


def write_e2e_trace(path: str, step_host, torch):
    """One ffpp_run_host call under torch.profiler (CUPTI activity records): every copy, memset and kernel with its
    stream, start and duration, as text.  A diagnostic, never a timing source for the bench line."""
    from torch.profiler import ProfilerActivity, profile
    import tempfile
    with profile(activities=[ProfilerActivity.CUDA]) as prof:
        step_host()
        torch.cuda.synchronize()
    with tempfile.NamedTemporaryFile(suffix=".json") as tf:
        prof.export_chrome_trace(tf.name)
        ev = [e for e in json.load(open(tf.name))["traceEvents"] if e.get("ph") == "X" and e.get("cat") in ("kernel", "gpu_memcpy", "gpu_memset")]
    ev.sort(key=lambda e: e["ts"])
    t0 = ev[0]["ts"] if ev else 0
    with open(path, "w") as fh:
        fh.write("start_us  dur_us  end_us  stream  what  bytes\n")
        for e in ev:
            fh.write(f"{e['ts'] - t0:9.1f} {e['dur']:8.1f} {e['ts'] - t0 + e['dur']:9.1f}  s{e['args'].get('stream', '?'):<3} "
                     f"{e['name'].replace('void ffpp::', '')[:40]:40s} {e['args'].get('bytes', '')}\n")


def a3_roofline(work: np.ndarray, ms: float, sm_count: int, sm_mhz: float) -> dict:
    """Method's own fp32 lane-instructions of one a3 launch (device-counted) against the fp32 lane peak."""
    ops = A3_OPS_PER_EXACT_IOU * int(work[1])
    peak = sm_count * FP32_LANES_PER_SM * sm_mhz * 1e6
    ach = ops / (ms * 1e-3)
    return {"bound": "alu", "achieved": ach / 1e12, "peak": peak / 1e12, "unit": "T fp32 lane-instr/s", "frac": ach / peak,
            "counted_work": {"exact_ious": int(work[1]), "edges": int(work[2]),
                             "frames_on_overflow_path": int(work[3]), "lane_instructions": ops,
                             "how": "device counters of the counting instantiation of the a3 kernel, separate untimed run "
                                    f"(ffpp_debug_count_work); {A3_OPS_PER_EXACT_IOU} per exact IoU"},
            "peak_source": f"{sm_count} SM x {FP32_LANES_PER_SM} fp32 lanes x {sm_mhz:.0f} MHz (sm_count from the handle, clocks.max.sm)"}


# --------------------------------------------------------------------------------------------------------------
# one config on this rank's GPU
# --------------------------------------------------------------------------------------------------------------
class Bench:
    def __init__(self, c: int, rank: int, flush, stream):
        import torch
        import flockgen
        import paper_2512_07009_b200 as ffpp
        self.torch, self.ffpp = torch, ffpp
        self.c = c
        self.w = flockgen.make_config(c, seed_offset=rank)
        self.pp = ffpp.FFPP.for_workload(self.w)
        self.info = self.pp.info()
        self.stream = stream
        self.flush = flush
        self.raw_pinned = torch.from_numpy(self.w.raw).pin_memory()
        self.raw_dev = self.raw_pinned.cuda(non_blocking=False)
        self.out = self.pp.alloc_outputs(self.w.B, self.w.frame_dims)

    def step(self):
        self.pp.run(self.raw_dev, self.w.N_per_frame, self.w.frame_dims, out=self.out, stream=self.stream)

    def flush_l2(self, clean: bool = True):
        """Outside every event pair.  512 MB write evicts the whole L2; the 512 MB read that follows replaces the dirty
        lines of that write with clean ones (cold AND clean: nothing is being written back while the step runs)."""
        self.flush.zero_()
        if clean:
            self.pp.stream_read(self.flush, self.stream)

    def timed_steps(self, steps: int, clean: bool = True) -> np.ndarray:
        torch = self.torch
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for k in range(steps):
            self.flush_l2(clean)
            ev[k][0].record(self.stream)
            self.step()
            ev[k][1].record(self.stream)
        torch.cuda.synchronize()
        return np.array([a.elapsed_time(b) for a, b in ev], dtype=np.float64)

    def stage_ms(self, iters: int, mode: str) -> np.ndarray:
        """Per-stage durations from the library's own events on the launching stream.  mode: cold_clean | cold_dirty | warm."""
        torch = self.torch
        self.pp.set_stage_timing(True)
        acc = []
        for i in range(iters + (2 if mode == "warm" else 0)):
            if mode != "warm":
                self.flush_l2(mode == "cold_clean")
            self.step()
            torch.cuda.synchronize()
            acc.append(self.pp.stage_ms().astype(np.float64))
        self.pp.set_stage_timing(False)
        return np.mean(np.stack(acc[2:] if mode == "warm" else acc), axis=0)

    def read_floor_ms(self, clean: bool) -> float:
        torch = self.torch
        rd = []
        for _ in range(8):
            self.flush_l2(clean)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(self.stream); self.pp.stream_read(self.raw_dev, self.stream); e1.record(self.stream)
            torch.cuda.synchronize()
            rd.append(e0.elapsed_time(e1))
        return float(np.median(rd[2:]))

    def counted_work(self) -> np.ndarray:
        self.pp.count_work(True)
        self.step()
        self.torch.cuda.synchronize()
        work = self.pp.debug_read(4, self.w.B)
        self.pp.count_work(False)
        self.step()
        self.torch.cuda.synchronize()
        return work

    def alg_bytes(self, n_surv, n_sorted, kept):
        w = self.w
        elem = 2 if w.params["dtype"] == "fp16" else 4
        key_b = self.info.key_bits // 8
        row_b = 5 * elem
        cells = int(self.out.density_offsets[-1])
        n_sv, n_in, kept_n = int(n_surv.sum()), int(n_sorted.sum()), int(kept.sum())
        return {
            "a1_threshold_compact": w.total_candidates * row_b + n_sv * key_b,   # read every row once, write one key per survivor
            "a2_select_decode_bin": n_sv * key_b + n_in * (row_b + 36),          # read keys, gather top-K rows, write box + culling box + key
            "a4_nms_resolve_emit": n_in * 24 + kept_n * 24 + 4 * w.B,            # read top-K records, write kept records + counts
            "a5a6_density": 4 * cells + 2 * cells + 16 * kept_n,                # histogram read, every density cell written once, kept boxes read
        }, row_b, cells


def quick_config(c: int, rank: int, flush, stream, hbm_peak: float) -> dict:
    """Configs other than the main one: a short cold-clean measurement for the `configs` block."""
    b = Bench(c, rank, flush, stream)
    for _ in range(3):
        b.flush_l2(); b.step()
    b.torch.cuda.synchronize()
    B = b.w.B
    n_sorted, n_surv = b.pp.debug_read(1, B), b.pp.debug_read(0, B)
    kept = b.out.counts_numpy().astype(np.int64)
    step_ms = b.timed_steps(10)
    st = b.stage_ms(5, "cold_clean")
    ab, _, _ = b.alg_bytes(n_surv, n_sorted, kept)
    ms = float(np.mean(step_ms))
    res = {"workload": CONFIG_DESC[c], "ms_per_step": ms, "frames_per_s": B / (ms * 1e-3), "candidates_per_s": b.w.total_candidates / (ms * 1e-3),
           "a1_frac_of_hbm_peak": ab["a1_threshold_compact"] / (st[1] * 1e-3) / 1e9 / hbm_peak,
           "a6_frac_of_hbm_peak": ab["a5a6_density"] / (st[5] * 1e-3) / 1e9 / hbm_peak,
           "stages_ms": {nm: float(st[i]) for i, nm in enumerate(b.ffpp.STAGE_NAMES)}, "steps": 10,
           "kept": int(kept.sum()), "entering_nms": int(n_sorted.sum())}
    b.pp.close()
    return res



# --------------------------------------------------------------------------------------------------------------
# SURVEY §8(f) rows f1-f4 (include/ffpp_next.h): short cold-L2 measurements, reported beside the hot path
# --------------------------------------------------------------------------------------------------------------
def next_rows(b: "Bench", hbm_peak: float) -> dict:
    import flockgen
    torch, ffpp, pp, w, out = b.torch, b.ffpp, b.pp, b.w, b.out
    stream = b.stream

    def timed(fn, iters=8):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(iters):
            b.flush_l2()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts))

    res = {}
    b.step(); torch.cuda.synchronize()
    cells = int(out.density_offsets[-1])
    B = w.B
    # f1: entropy, clustering degree, threshold + connected components on this batch's own density grids
    MAXR = 512
    h_ent = torch.empty(B, dtype=torch.float64, device="cuda"); h_deg = torch.empty(B, dtype=torch.float64, device="cuda")
    h_lab = torch.empty(cells, dtype=torch.int32, device="cuda"); h_reg = torch.zeros((B, MAXR, 8), dtype=torch.int32, device="cuda")
    h_cnt = torch.empty(B, dtype=torch.int32, device="cuda")
    dims = np.ascontiguousarray(w.frame_dims, dtype=np.int32).reshape(-1, 2)

    def f1():
        rc = pp._lib.ffpp_heatmap_stats(pp._h, out.density.data_ptr(), B, dims.ctypes.data, 0.05, 4, MAXR, stream.cuda_stream,
                                        h_ent.data_ptr(), h_deg.data_ptr(), h_lab.data_ptr(), h_reg.data_ptr(), h_cnt.data_ptr())
        assert rc == 0, pp.last_error()
    ms = timed(f1)
    byt = 8 * cells + 32 * int(h_cnt.clamp(max=MAXR).sum())
    res["f1_heatmap_stats"] = {"ms": ms, "workload": f"{B} density grids of this batch ({cells} cells), threshold 0.05, 4-connectivity",
                               "regions": int(h_cnt.sum()), "mean_entropy_nats": float(h_ent.mean()), "mean_clustering_degree": float(h_deg.mean()),
                               "algorithmic_bytes": byt, "GB/s": byt / (ms * 1e-3) / 1e9, "frac_of_hbm_peak": byt / (ms * 1e-3) / 1e9 / hbm_peak,
                               "bytes_note": "4 B per cell read + 4 B per cell of label image written + 32 B per region",
                               "kernels": "ke_partial ke_final kc_init kc_merge kc_flatten kr_count_place kr_scan kr_count_place kc_stats kc_final"}
    # f2: exact-position density of the kept boxes, and what the binning of A14 costs against it
    d_ex = torch.empty(cells, dtype=torch.float32, device="cuda")

    def f2():
        rc = pp._lib.ffpp_density_exact(pp._h, out.boxes.data_ptr(), out.counts.data_ptr(), B, dims.ctypes.data, stream.cuda_stream, d_ex.data_ptr())
        assert rc == 0, pp.last_error()
    ms = timed(f2)
    diff = (d_ex - out.density).abs()
    kept = int(out.counts.sum())
    R = int(b.info.radius)
    evals = kept * (2 * R + 1) ** 2
    res["f2_density_exact"] = {"ms": ms, "workload": f"kept boxes of this batch ({kept}) onto {cells} cells", "cells_per_s": cells / (ms * 1e-3),
                               "kernel_evaluations_needed": evals, "Gevals/s": evals / (ms * 1e-3) / 1e9,
                               "binning_error_of_A14": {"max_abs": float(diff.max()), "mean_abs": float(diff.mean()),
                                                        "max_density": float(d_ex.max()), "note": "|binned out_density - exact-position density| per cell (interior and border: the exact form has no fold)"},
                               "kernels": "kd_exact"}
    # f3: segmentation-mask post-processing, 8 masks of 1920x1080 fp16
    MB, MW, MH, MAXC = 8, 1920, 1080, 4096
    masks = torch.from_numpy(flockgen.make_mask_batch(MB, MW, MH, birds=800, seed=5)).cuda()
    m_lab = torch.empty((MB, MH, MW), dtype=torch.int32, device="cuda"); m_tab = torch.zeros((MB, MAXC, 8), dtype=torch.int32, device="cuda")
    m_cnt = torch.empty(MB, dtype=torch.int32, device="cuda")

    def f3():
        rc = pp._lib.ffpp_mask_components(pp._h, masks.data_ptr(), 1, MB, MW, MH, 0.5, 8, 20, MAXC, stream.cuda_stream, m_lab.data_ptr(),
                                          m_tab.data_ptr(), m_cnt.data_ptr())
        assert rc == 0, pp.last_error()
    ms = timed(f3)
    byt = 6 * MB * MW * MH
    res["f3_mask_components"] = {"ms": ms, "ms_per_frame": ms / MB, "frames_per_s": MB / (ms * 1e-3),
                                 "workload": f"{MB} synthetic 1920x1080 fp16 bird masks (~800 blobs each), threshold 0.5, 8-connectivity, min_area 20",
                                 "components": int(m_cnt.sum()), "algorithmic_bytes": byt, "GB/s": byt / (ms * 1e-3) / 1e9,
                                 "frac_of_hbm_peak": byt / (ms * 1e-3) / 1e9 / hbm_peak, "bytes_note": "2 B per pixel read + 4 B per pixel of label image written",
                                 "paper_context": "paper: 40.2 -> 11.4 ms per frame on the CPU of a g4dn.2xlarge (PAPER.md:L151)",
                                 "kernels": "kc_init kc_merge kc_flatten kr_count_place kr_scan kr_count_place kc_stats kc_final"}
    del masks, m_lab
    # f4: pre-processing, 8 frames of 1920x1080 -> 640x640 fp16 CHW, alone and overlapped with ffpp_run on a second stream
    imgs = torch.from_numpy(flockgen.make_image_batch(MB, MW, MH, seed=5)).cuda()
    dst = torch.empty((MB, 3, 640, 640), dtype=torch.float16, device="cuda")
    mean = np.array([0.485, 0.456, 0.406], dtype=np.float32); std = np.array([0.229, 0.224, 0.225], dtype=np.float32)
    lib = ffpp.load_library()

    def f4(st=stream):
        rc = lib.ffpp_preprocess(imgs.data_ptr(), MB, MH, MW, 640, 640, mean.ctypes.data, std.ctypes.data, 1, st.cuda_stream, dst.data_ptr())
        assert rc == 0
    ms = timed(f4)
    byt = imgs.numel() + dst.numel() * 2
    side = torch.cuda.Stream()

    def serial():
        f4(); b.step()

    def overlapped():
        side.wait_stream(stream)
        f4(side)
        b.step()
        stream.wait_stream(side)
    ms_serial, ms_overlap = timed(serial), timed(overlapped)
    res["f4_preprocess"] = {"ms": ms, "ms_per_frame": ms / MB, "workload": f"{MB} frames 1920x1080x3 uint8 -> 640x640 fp16 CHW, ImageNet mean/std",
                            "algorithmic_bytes": byt, "GB/s": byt / (ms * 1e-3) / 1e9, "frac_of_hbm_peak": byt / (ms * 1e-3) / 1e9 / hbm_peak,
                            "bytes_note": "3 B per source pixel read once + 6 B per destination pixel written",
                            "stream_overlap": {"ms_preprocess_then_ffpp_run_one_stream": ms_serial, "ms_preprocess_on_second_stream": ms_overlap,
                                               "note": "next batch's pre-processing on a second stream while this batch's ffpp_run runs (PAPER.md:L308-310)"},
                            "paper_context": "paper: 8.8 ms per frame (PAPER.md:L151)", "kernels": "kp_preprocess"}
    return res

# --------------------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2512_07009_b200 as ffpp

    rank, local_rank, world = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    ffpp.load_library()
    hbm_peak, peak_src, sm_max_mhz = load_peaks()

    c = args.config
    stream = torch.cuda.current_stream()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    b = Bench(c, rank, flush, stream)
    w, pp, info, out = b.w, b.pp, b.info, b.out
    B, total_cand = w.B, w.total_candidates
    sm_count = int(info.sm_count)

    def barrier():
        if world > 1:
            dist.barrier()

    # ---- warm-up ----
    W = max(args.warmup, 3)
    for _ in range(W):
        b.flush_l2(); b.step()
    torch.cuda.synchronize()
    n_sorted = pp.debug_read(1, B)
    n_surv = pp.debug_read(0, B)
    kept = out.counts_numpy().astype(np.int64)
    pairs = pair_count(n_sorted)

    # ---- timed: device-resident inputs, cold and clean L2 ----
    sampler = ClockSampler(local_rank)
    barrier(); torch.cuda.synchronize()
    sampler.start()
    t_wall0 = time.perf_counter()
    step_ms = b.timed_steps(args.steps)
    torch.cuda.synchronize(); barrier()
    t_wall = time.perf_counter() - t_wall0
    total_ms = float(step_ms.sum())

    # ---- per-stage durations (library's own events on the launching stream), same launch configuration ----
    n_it = min(max(args.steps, 3), 20)
    stage_ms = b.stage_ms(n_it, "cold_clean")
    dirty_ms = b.stage_ms(n_it, "cold_dirty")
    warm_ms = b.stage_ms(n_it, "warm")
    read_clean_ms = b.read_floor_ms(True)
    read_dirty_ms = b.read_floor_ms(False)
    work = b.counted_work()                 # separate, untimed: the counting instantiation of the a3 kernel

    # ---- e2e: host buffers through ffpp_run_host ----
    cells = int(out.density_offsets[-1])
    h_boxes = torch.empty((B, pp.top_k, 6), dtype=torch.float32).pin_memory()
    h_counts = torch.empty((B,), dtype=torch.int32).pin_memory()
    h_density = torch.empty((cells,), dtype=torch.float32).pin_memory()
    hout = ffpp.Output()
    hout.boxes, hout.counts, hout.density, hout.density_offsets = h_boxes, h_counts, h_density, out.density_offsets

    def step_host():
        pp.run_host(b.raw_pinned, w.N_per_frame, w.frame_dims, out=hout, stream=stream)

    e2e_steps = args.steps
    for _ in range(3):
        step_host()
    barrier(); torch.cuda.synchronize()
    t_e2e = 0.0
    for _ in range(e2e_steps):
        b.flush_l2(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        step_host()
        t_e2e += time.perf_counter() - t0
    torch.cuda.synchronize(); barrier()
    clocks = sampler.stop()
    if args.e2e_trace and rank == 0:
        write_e2e_trace(args.e2e_trace, step_host, torch)
    h2d = int(w.raw.nbytes)
    d2h = int(4 * B + 4 * cells + 24 * int(kept.sum()))
    # PCIe floor of the same transfers: pinned H2D of the raw buffer and pinned D2H of the density, each alone
    def copy_ms(dst, src):
        ts = []
        for _ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); dst.copy_(src, non_blocking=True); e1.record(stream)
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        return float(np.median(ts[1:]))
    h2d_ms = copy_ms(b.raw_dev, b.raw_pinned)
    d2h_ms = copy_ms(h_density, out.density) * (d2h / max(4 * cells, 1))

    # ---- the other configs (single-GPU default run only): short cold-clean measurements ----
    configs = {}
    if world == 1 and not args.no_other_configs:
        for cc in (1, 2, 3, 4, 5):
            if cc != c:
                try:
                    configs[str(cc)] = quick_config(cc, rank, flush, stream, hbm_peak)
                except Exception as exc:           # reported, never fatal for the main line
                    configs[str(cc)] = {"workload": CONFIG_DESC[cc], "error": str(exc)}

    # ---- SURVEY §8(f) rows f1-f4 (single-GPU default run only) ----
    nxt = {}
    if world == 1 and not args.no_next:
        try:
            nxt = next_rows(b, hbm_peak)
        except Exception as exc:                   # reported, never fatal for the main line
            nxt = {"error": str(exc)}

    # ---- reduce over ranks ----
    total_ms, t_e2e, frames_all, cand_all = reduce_over_ranks(total_ms, t_e2e, float(B), float(total_cand), world, "cuda")

    if rank == 0:
        K = args.steps
        fps = frames_all * K / (total_ms * 1e-3)
        cps = cand_all * K / (total_ms * 1e-3)
        kept_n = int(kept.sum())
        alg_bytes, row_b, _ = b.alg_bytes(n_surv, n_sorted, kept)
        cell_b = 4 * cells
        stages = {}
        names = ffpp.STAGE_NAMES
        for i, nm in enumerate(names):
            stages[nm] = {"ms": float(stage_ms[i]), "share_of_step": float(stage_ms[i] / stage_ms.sum()), "kernels": ffpp.STAGE_KERNELS[nm],
                          "ms_cold_dirty": float(dirty_ms[i]), "ms_warm": float(warm_ms[i])}
            if nm in alg_bytes:
                gbs = alg_bytes[nm] / (stage_ms[i] * 1e-3) / 1e9
                stages[nm].update({"algorithmic_bytes": alg_bytes[nm], "GB/s": gbs, "frac_of_hbm_peak": gbs / hbm_peak})
        s1 = stages["a1_threshold_compact"]
        raw_bytes = total_cand * row_b
        s1["plain_read_of_same_bytes"] = {
            "ms": read_clean_ms, "GB/s": raw_bytes / (read_clean_ms * 1e-3) / 1e9, "frac_of_hbm_peak": raw_bytes / (read_clean_ms * 1e-3) / 1e9 / hbm_peak,
            "ms_cold_dirty": read_dirty_ms,
            "note": "k0_stream_read over the raw head output under the same cold-clean regime: what a pure read of this many bytes reaches"}
        s1["frac_of_plain_read"] = read_clean_ms / float(stage_ms[1])
        s3 = stages["a3_nms_pairs"]
        s3["iou_pairs_decided"] = pairs
        s3["Gpairs/s_decided"] = pairs / (stage_ms[3] * 1e-3) / 1e9
        r3 = a3_roofline(work, float(stage_ms[3]), sm_count, sm_max_mhz)
        # speed-up over the all-pairs bitmask method at ITS ALU ceiling (context, not a roofline fraction)
        allpairs_ceiling = sm_count * FP32_LANES_PER_SM * sm_max_mhz * 1e6 / A3_OPS_PER_EXACT_IOU
        s3["dense_equiv_speedup"] = (pairs / (stage_ms[3] * 1e-3)) / allpairs_ceiling
        s3["alu"] = {k: r3[k] for k in ("achieved", "peak", "unit", "frac", "counted_work")}
        # dominant kernel = the stage with the largest share of the step
        dom = int(np.argmax(stage_ms[1:])) + 1
        if dom == 3:
            roofline = dict(r3)
            roofline["dense_equiv_speedup"] = s3["dense_equiv_speedup"]
        else:
            sd = stages[names[dom]]
            roofline = {"bound": "hbm", "achieved": sd["GB/s"], "peak": hbm_peak, "unit": "GB/s", "frac": sd["GB/s"] / hbm_peak, "peak_source": peak_src}
        roofline["kernel"] = ffpp.STAGE_KERNELS[names[dom]]
        roofline["stage"] = names[dom]
        roofline["avg_launch_ms"] = float(stage_ms[dom])
        roofline["traffic"] = None
        tr_path = os.path.join(ROOT, "profiles", f"r2_traffic_config{c}.csv")
        if os.path.exists(tr_path):      # STATIC: per-launch numbers of the committed ncu --set full capture of this config
            import csv
            with open(tr_path, newline="") as fh:
                rows = {r["kernel"]: r for r in csv.DictReader(fh)}
            k = rows.get(roofline["kernel"].split(" ")[0])
            if k:
                k = {kk: float(vv) for kk, vv in k.items() if kk != "kernel"}
                roofline["traffic"] = k["dram_bytes"]            # dram__bytes_read.sum + dram__bytes_write.sum
                roofline["static_from_ncu_capture"] = {
                    "source": f"profiles/r2_traffic_config{c}.csv (one ncu --set full launch of the committed build; NOT measured by this run)",
                    **{kk: k[kk] for kk in k if kk != "dram_bytes"}}
        # whole step against HBM: bytes the path must move (raw in, three outputs out) / device step time
        step_bytes = total_cand * row_b + 24 * kept_n + 4 * B + cell_b
        step_gbs = step_bytes / (float(np.median(step_ms)) * 1e-3) / 1e9
        step_roofline = {"bound": "hbm", "algorithmic_bytes": step_bytes, "achieved": step_gbs, "peak": hbm_peak, "unit": "GB/s",
                         "frac": step_gbs / hbm_peak, "note": "raw head output read once + kept boxes, counts and density written once, "
                         "over the median device step time of this rank; every intermediate is overhead against this bound"}

        # ---- CPU baseline: the oracle as it stands on this box's host cores, bounded sample ----
        try:
            t_cpu, nf, rows = oracle_time(w, CPU_BASELINE_FRAMES[c])
            cpu = {"value": nf / t_cpu, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": f"first {nf} of {B} frames of {w.name} ({rows} candidates), one pass, single thread, {t_cpu:.2f} s",
                   "candidates_per_s": rows / t_cpu, "host_cpus": os.cpu_count()}
        except Exception as exc:  # the baseline is reported, never required for the GPU numbers
            cpu = {"value": None, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": f"failed: {exc}"}

        ms_step = total_ms / K
        configs[str(c)] = {"workload": CONFIG_DESC[c], "ms_per_step": ms_step, "frames_per_s": B / (ms_step * 1e-3),
                           "candidates_per_s": total_cand / (ms_step * 1e-3),
                           "a1_frac_of_hbm_peak": stages["a1_threshold_compact"]["frac_of_hbm_peak"],
                           "a6_frac_of_hbm_peak": stages["a5a6_density"]["frac_of_hbm_peak"],
                           "stages_ms": {nm: float(stage_ms[i]) for i, nm in enumerate(names)}, "steps": K,
                           "kept": kept_n, "entering_nms": int(n_sorted.sum())}
        e2e_ms = 1e3 * t_e2e / e2e_steps
        line = {
            "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "input_dtype": w.params["dtype"], "data": "synthetic",
            "config": {"workload": CONFIG_DESC[c], "frames_per_step_per_gpu": B, "candidates_per_step_per_gpu": total_cand,
                       "input_dtype": w.params["dtype"], "top_k": w.params["top_k"], "conf": w.params["conf_thresh"],
                       "iou": w.params["iou_thresh"], "sigma_cells": w.params["sigma_cells"],
                       "l2": "cold and clean between steps (512 MB write, then 512 MB read, outside the event pair)",
                       "seed": "config_seed(c)+rank"},
            "candidates_per_s": cps,
            "step_ms_min": float(step_ms.min()), "step_ms_median": float(np.median(step_ms)), "wall_s_timed_loop": t_wall,
            "e2e": {"value": frames_all * e2e_steps / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms, "candidates_per_s": cand_all * e2e_steps / t_e2e,
                    "pcie_floor_ms": max(h2d_ms, d2h_ms), "pcie_h2d_ms": h2d_ms, "pcie_d2h_ms": d2h_ms,
                    "pcie_h2d_GB/s": h2d / (h2d_ms * 1e-3) / 1e9, "frac_of_pcie_floor": max(h2d_ms, d2h_ms) / e2e_ms,
                    "api": "ffpp_run_host (pinned host buffers, copies + sync inside the timed region)"},
            "gpu_launches": ffpp.LAUNCHES_PER_RUN * K,
            "launches_per_step": {"kernels": ffpp.LAUNCHES_PER_RUN, "memsets": 0, "descriptor_uploads": 0},
            "roofline": roofline,
            "step_roofline": step_roofline,
            "stages": stages,
            "warm_l2": {"ms_per_step": float(warm_ms.sum()), "frames_per_s": B / (float(warm_ms.sum()) * 1e-3),
                        "note": "no L2 flush between steps: inputs of <= 126 MB are served from L2, so a1's GB/s is not an HBM figure"},
            "cold_dirty_l2": {"ms_per_step": float(dirty_ms.sum()),
                              "note": "512 MB write only (round 1's regime): the first kernels compete with the write-back of dirty lines"},
            "configs": configs,
            "next_rows": nxt,
            "cpu_baseline": cpu,
            "clocks": clocks,
            "workload_stats": {"survivors": int(n_surv.sum()), "entering_nms": int(n_sorted.sum()), "kept": kept_n,
                               "iou_pairs": pairs, "density_cells": cells, "workspace_bytes": int(info.workspace_bytes)},
            "paper_context": "paper: up to 2x pipeline speedup on AWS g4dn.2xlarge (T4), $0.69 -> $0.31 per run; no number for this path",
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short measurements of the other four configs")
    ap.add_argument("--no-next", action="store_true", help="skip the measurements of the SURVEY 8(f) rows f1-f4")
    ap.add_argument("--e2e-trace", default=None, metavar="FILE",
                    help="also write a text timeline (copies and kernels per stream, from torch.profiler / CUPTI) of one ffpp_run_host call")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
