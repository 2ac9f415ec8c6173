"""Element-by-element comparison of the CUDA path with the oracle (BASELINE.json north_star parity bar):
kept index lists and decoded boxes bit-exact, sigmoid scores within 1e-6, density within
max(1e-5, 1e-4*|ref|) per cell plus the grid-sum invariant."""
import numpy as np


def compare(out, ref, w, *, check_stage=None):
    """out: paper_2512_07009_b200.Output (device or host); ref: oracle.Result; w: flockgen.Workload-like."""
    B = len(w.N_per_frame)
    counts = out.counts_numpy()
    boxes = out.boxes_numpy()
    dens = out.density_numpy()
    assert counts.shape == (B,)
    assert np.array_equal(counts, ref.counts), f"kept counts differ: {counts.tolist()[:8]} vs {ref.counts.tolist()[:8]}"
    for f in range(B):
        n = int(ref.counts[f])
        g, o = boxes[f, :n], ref.boxes[f, :n]
        assert np.array_equal(g["cand_index"], o["cand_index"]), f"frame {f}: kept index lists differ"
        for k in ("x1", "y1", "x2", "y2"):
            assert np.array_equal(g[k].view(np.uint32), o[k].view(np.uint32)), f"frame {f}: decoded {k} not bit-exact"
        if n:
            assert np.max(np.abs(g["score"] - o["score"])) <= 1e-6, f"frame {f}: sigmoid score"
    assert dens.shape == ref.density.shape
    tol = np.maximum(1e-5, 1e-4 * np.abs(ref.density))
    bad = np.abs(dens - ref.density) > tol
    assert not bad.any(), f"density: {int(bad.sum())} cells out of tolerance, max err {np.abs(dens - ref.density).max()}"
    dims = np.asarray(w.frame_dims).reshape(-1, 2)
    off = ref.density_offsets
    for f in range(B):
        b = boxes[f, :int(ref.counts[f])]
        cx = (b["x1"] + b["x2"]) * np.float32(0.5)
        cy = (b["y1"] + b["y2"]) * np.float32(0.5)
        n_in = int(((cx >= 0) & (cx < dims[f, 0]) & (cy >= 0) & (cy < dims[f, 1])).sum())
        s = float(dens[off[f]:off[f + 1]].astype(np.float64).sum())
        assert abs(s - n_in) <= 1e-4 * max(n_in, 1), f"frame {f}: grid sum {s} vs {n_in} in-frame kept"
    if check_stage is not None:
        pp = check_stage
        assert np.array_equal(pp.debug_read(0, B), ref.survivor_counts), "survivor counts after threshold"
        assert np.array_equal(pp.debug_read(1, B), ref.sorted_counts), "sorted counts"
        assert np.array_equal(pp.debug_read(2, B), ref.sorted_idx), "sorted candidate index lists"
