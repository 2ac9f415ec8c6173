"""GPU parity of the SURVEY §8(f) rows f1-f4 (include/ffpp_next.h) against oracle/ffpp_next_oracle.cpp, through the C ABI.
Inputs never come from the CUDA path: density grids and kept boxes fed to f1 / f2 are the ORACLE's (uploaded), masks
and images are flockgen's.  Bars: labels, region tables (label, area, bounding box) and counts bit-exact; masses and
scores within 1e-6 relative; entropy / clustering degree within 1e-9 absolute (double on both sides); exact-position
density within max(1e-5, 1e-4 |ref|) per cell (the hot path's A20 bar); pre-processing within 2e-6 absolute in fp32 and
one fp16 rounding (2^-11 relative + 1e-6) in fp16."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(oracle_mod, gen_mod):
    import torch
    import paper_2512_07009_b200 as m
    assert torch.cuda.is_available()
    m.load_library()
    return torch, m, oracle_mod, gen_mod


def check_regions(got_tab, got_n, ref_tab, ref_n, what):
    assert got_n == ref_n, f"{what}: region count {got_n} vs {ref_n}"
    k = len(ref_tab)
    g = got_tab[:k]
    for fld in ("label", "area", "x0", "y0", "x1", "y1"):
        assert np.array_equal(g[fld], ref_tab[fld]), f"{what}: {fld}"
    np.testing.assert_allclose(g["mass"], ref_tab["mass"], rtol=1e-6, atol=1e-7, err_msg=what)


# ---------------------------------------------------------------- f1
@pytest.mark.parametrize("cfg,B,conn,thr", [(1, None, 4, 0.02), (2, None, 8, 0.03), (3, 4, 4, 0.05), (4, 4, 4, 0.08), (5, 8, 4, 0.04), (5, 8, 8, 0.15)])
def test_heatmap_stats_matches_the_oracle(env, cfg, B, conn, thr):
    torch, m, oracle, gen = env
    w = gen.make_config(cfg) if B is None else gen.make_config(cfg, B=B)
    ref = oracle.run(w.params, w.raw, w.N_per_frame, w.frame_dims)            # the ORACLE's density grids are the input
    pp = m.FFPP.for_workload(w)
    dens = torch.from_numpy(ref.density).cuda()
    MAXR = 512
    res = pp.heatmap_stats(dens, w.frame_dims, thr, connectivity=conn, max_regions=MAXR)
    torch.cuda.synchronize()
    ent, deg = res["entropy"].cpu().numpy(), res["degree"].cpu().numpy()
    labels = res["labels"].cpu().numpy()
    tabs = m.regions_numpy(res["regions"])
    counts = res["region_counts"].cpu().numpy()
    off = ref.density_offsets
    dims = np.asarray(w.frame_dims).reshape(-1, 2)
    nonempty = 0
    for f in range(w.B):
        gw, gh = dims[f, 0] // 8, dims[f, 1] // 8
        D = ref.density[off[f]:off[f + 1]].reshape(gh, gw)
        assert abs(ent[f] - oracle.entropy(D)) <= 1e-9, f"frame {f}: entropy {ent[f]} vs {oracle.entropy(D)}"
        assert abs(deg[f] - oracle.clustering_degree(D)) <= 1e-9, f"frame {f}: clustering degree"
        lab, tab, n = oracle.regions(D, thr, conn=conn, max_regions=MAXR)
        assert np.array_equal(labels[off[f]:off[f + 1]].reshape(gh, gw), lab), f"frame {f}: label image"
        check_regions(tabs[f], int(counts[f]), tab, n, f"frame {f}")
        nonempty += n > 1
    assert nonempty >= max(1, w.B // 2), "thresholds of this test must cut the grids into several regions"


def test_heatmap_stats_edge_grids(env):
    """all-background, all-foreground (one region = whole grid), a threshold equal to a cell value (strict), table
    overflow (count reported beyond max_regions), an empty grid (entropy 0), and a replay on a cached geometry."""
    torch, m, oracle, gen = env
    params = dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=100, sigma_cells=2.0)
    dims = np.array([[640, 640], [320, 192], [64, 64]], dtype=np.int32)
    pp = m.FFPP(params, max_frames=3, max_total_candidates=8400 * 3, max_frame_w=640, max_frame_h=640)
    rng = np.random.default_rng(4)
    grids = [rng.random((80, 80)).astype(np.float32), np.zeros((24, 40), dtype=np.float32), np.full((8, 8), 0.5, dtype=np.float32)]
    grids[0][::2, ::2] = 2.0                                                   # 1600 isolated peaks above 1.5
    grids[0][1::2, :] = 0.0; grids[0][:, 1::2] = 0.0
    flat = np.concatenate([g.ravel() for g in grids])
    for thr, maxr in [(1.5, 64), (0.5, 16), (-1.0, 16), (0.25, 2048)]:
        res = pp.heatmap_stats(torch.from_numpy(flat).cuda(), dims, thr, connectivity=4, max_regions=maxr)
        torch.cuda.synchronize()
        tabs = m.regions_numpy(res["regions"]); counts = res["region_counts"].cpu().numpy(); labels = res["labels"].cpu().numpy()
        o = 0
        for f, g in enumerate(grids):
            lab, tab, n = oracle.regions(g, thr, conn=4, max_regions=maxr)
            assert np.array_equal(labels[o:o + g.size].reshape(g.shape), lab)
            check_regions(tabs[f], int(counts[f]), tab, n, f"thr {thr} grid {f}")
            assert abs(float(res["entropy"][f]) - oracle.entropy(g)) <= 1e-9
            assert abs(float(res["degree"][f]) - oracle.clustering_degree(g)) <= 1e-9
            o += g.size
    assert int(counts[0]) == 1600 and float(res["entropy"][1]) == 0.0 and float(res["degree"][1]) == 0.0


# ---------------------------------------------------------------- f2
@pytest.mark.parametrize("cfg,B", [(1, None), (2, 4), (3, 2), (4, 1), (5, 4)])
def test_density_exact_matches_the_oracle(env, cfg, B):
    torch, m, oracle, gen = env
    w = gen.make_config(cfg) if B is None else gen.make_config(cfg, B=B)
    ref = oracle.run(w.params, w.raw, w.N_per_frame, w.frame_dims)            # the ORACLE's kept boxes are the input
    pp = m.FFPP.for_workload(w)
    out = m.Output()
    out.boxes = torch.from_numpy(np.ascontiguousarray(ref.boxes).view(np.float32).reshape(w.B, pp.top_k, 6)).cuda()
    out.counts = torch.from_numpy(ref.counts).cuda()
    dens = pp.density_exact(out, w.frame_dims)
    torch.cuda.synchronize()
    got = dens.cpu().numpy()
    off = ref.density_offsets
    dims = np.asarray(w.frame_dims).reshape(-1, 2)
    p = w.params
    for f in range(w.B):
        b = ref.boxes[f, :int(ref.counts[f])]
        bx = np.stack([b["x1"], b["y1"], b["x2"], b["y2"]], 1)
        want, n_in = oracle.density_exact(bx, int(dims[f, 0]), int(dims[f, 1]), p.get("cell_px", 8), p["sigma_cells"], p.get("truncate_sigmas", 3.0))
        g = got[off[f]:off[f + 1]].reshape(want.shape)
        bad = np.abs(g - want) > np.maximum(1e-5, 1e-4 * np.abs(want))
        assert not bad.any(), f"frame {f}: {int(bad.sum())} cells out of tolerance, max err {np.abs(g - want).max()}"
        assert n_in > 0


def test_density_exact_hand_cases(env):
    """centroid on a cell centre reproduces the binned grid of ffpp_run's definition (G1); a centroid whose offset to a
    column of cell centres is exactly R is inside (<=), one fp32 step further is outside; out-of-frame centroids add nothing."""
    torch, m, oracle, gen = env
    params = dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=8, sigma_cells=2.0)
    pp = m.FFPP(params, max_frames=1, max_total_candidates=8400, max_frame_w=640, max_frame_h=640)
    cases = [[[304, 304, 344, 344]],                                           # (324, 324): cell centre
             [[300, 304, 340, 344]],                                           # u = 40.0: dx = +-6.5 .. -> |dx| <= 6 picks 12 columns
             [[308, 300, 348, 340], [-30, 100, 10, 140], [630, 630, 660, 660], [0, 0, 8, 8]],
             [[304 + 2 ** -10, 304, 344 + 2 ** -10, 344]]]
    for boxes in cases:
        rec = np.zeros((1, 8, 6), dtype=np.float32)
        rec[0, :len(boxes), :4] = np.asarray(boxes, dtype=np.float32)
        out = m.Output()
        out.boxes = torch.from_numpy(rec).cuda()
        out.counts = torch.tensor([len(boxes)], dtype=torch.int32, device="cuda")
        got = pp.density_exact(out, [[640, 640]]).cpu().numpy().reshape(80, 80)
        want, _ = oracle.density_exact(np.asarray(boxes, dtype=np.float32), 640, 640, 8, 2.0)
        assert np.array_equal(got != 0, want != 0), "support of the truncated kernel differs"
        np.testing.assert_allclose(got, want, rtol=1e-4, atol=1e-7)


# ---------------------------------------------------------------- f3
@pytest.mark.parametrize("dtype,W,H,B,conn,min_area", [("fp16", 640, 360, 3, 8, 1), ("fp32", 320, 200, 2, 4, 1), ("fp16", 1920, 1080, 2, 8, 20),
                                                       ("fp16", 333, 77, 2, 8, 2)])
def test_mask_components_match_the_oracle(env, dtype, W, H, B, conn, min_area):
    torch, m, oracle, gen = env
    masks = gen.make_mask_batch(B, W, H, birds=W * H / 2500.0, seed=17 + W, dtype=dtype)
    params = dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=8, sigma_cells=2.0)
    pp = m.FFPP(params, max_frames=1, max_total_candidates=8400, max_frame_w=640, max_frame_h=640)
    MAXC = 2048
    res = pp.mask_components(torch.from_numpy(masks).cuda(), 0.5, connectivity=conn, min_area=min_area, max_components=MAXC)
    torch.cuda.synchronize()
    labels = res["labels"].cpu().numpy(); tabs = m.regions_numpy(res["components"]); counts = res["counts"].cpu().numpy()
    for b in range(B):
        lab, tab, n = oracle.mask_components(masks[b], 0.5, conn=conn, min_area=min_area, max_components=MAXC)
        assert n > 3
        assert np.array_equal(labels[b], lab), f"mask {b}: label image"
        check_regions(tabs[b], int(counts[b]), tab, n, f"mask {b}")


def test_mask_components_adversarial_shapes(env):
    """a spiral and a comb (long union-find chains, many late merges), a checkerboard (8-connected: one component;
    4-connected: every pixel its own), full and empty masks, a table smaller than the component count."""
    torch, m, oracle, gen = env
    H, W = 96, 128
    yy, xx = np.mgrid[0:H, 0:W]
    spiral = np.zeros((H, W), dtype=np.float32)
    x, y, dx, dy, seg = W // 2, H // 2, 1, 0, 2
    while 0 <= x < W and 0 <= y < H:
        for _ in range(seg):
            if 0 <= x < W and 0 <= y < H:
                spiral[y, x] = 1
            x += dx; y += dy
        dx, dy = -dy, dx
        seg += 2 if dy == 0 else 0
    comb = np.zeros((H, W), dtype=np.float32); comb[:, ::2] = 1; comb[H - 1, :] = 1
    checker = ((xx + yy) % 2).astype(np.float32)
    batch = np.stack([spiral, comb, checker, np.ones((H, W), np.float32), np.zeros((H, W), np.float32)])
    params = dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=8, sigma_cells=2.0)
    pp = m.FFPP(params, max_frames=1, max_total_candidates=8400, max_frame_w=640, max_frame_h=640)
    for conn, maxc in [(8, 64), (4, 64), (4, 8192)]:
        res = pp.mask_components(torch.from_numpy(batch).cuda(), 0.5, connectivity=conn, max_components=maxc)
        torch.cuda.synchronize()
        labels = res["labels"].cpu().numpy(); tabs = m.regions_numpy(res["components"]); counts = res["counts"].cpu().numpy()
        for b in range(len(batch)):
            lab, tab, n = oracle.mask_components(batch[b], 0.5, conn=conn, max_components=maxc)
            assert np.array_equal(labels[b], lab), f"conn {conn} mask {b}"
            check_regions(tabs[b], int(counts[b]), tab, n, f"conn {conn} mask {b}")
    assert int(counts[2]) == H * W // 2 and int(counts[3]) == 1 and int(counts[4]) == 0


# ---------------------------------------------------------------- f4
@pytest.mark.parametrize("src,dst,out_dtype", [((1080, 1920), (640, 640), "fp16"), ((720, 1280), (736, 1280), "fp32"), ((270, 480), (1088, 1920), "fp16"),
                                               ((97, 131), (53, 75), "fp32"), ((64, 64), (64, 64), "fp32")])
def test_preprocess_matches_the_oracle(env, src, dst, out_dtype):
    torch, m, oracle, gen = env
    B = 2
    imgs = gen.make_image_batch(B, src[1], src[0], seed=31 + src[0])
    mean, std = [0.485, 0.456, 0.406], [0.229, 0.224, 0.225]
    got = m.preprocess(torch.from_numpy(imgs).cuda(), dst[0], dst[1], mean, std, out_dtype=out_dtype)
    torch.cuda.synchronize()
    got = got.cpu().numpy().astype(np.float64)
    for b in range(B):
        want = oracle.preprocess(imgs[b], dst[0], dst[1], mean, std)
        err = np.abs(got[b] - want)
        tol = 2e-6 + 4e-7 * np.abs(want) if out_dtype == "fp32" else 1e-6 + 2.0 ** -11 * np.abs(want) * 1.001 + 2e-6
        assert (err <= tol).all(), f"image {b}: max err {err.max()} at {np.unravel_index(err.argmax(), err.shape)}"
