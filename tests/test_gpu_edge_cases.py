"""GPU edge cases: empty / tiny / boundary-size inputs, ties, ABI misuse."""
import numpy as np
import pytest

from parity import compare

pytestmark = pytest.mark.gpu

P = dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=3000, strides=[8, 16, 32], cell_px=8, sigma_cells=2.0,
         truncate_sigmas=3.0)


class W:
    def __init__(self, raw, dims, params):
        import flockgen
        self.raw = raw
        self.frame_dims = np.asarray(dims, dtype=np.int32).reshape(-1, 2)
        self.N_per_frame = np.array([flockgen.frame_candidates(int(a), int(b)) for a, b in self.frame_dims], dtype=np.int32)
        self.params = params
        assert raw.shape[0] == int(self.N_per_frame.sum())


@pytest.fixture(scope="module")
def env(oracle_mod, gen_mod):
    torch = pytest.importorskip("torch")
    assert torch.cuda.is_available()
    import paper_2512_07009_b200 as m
    m.load_library()
    return torch, m, oracle_mod, gen_mod


def check(env, w, **kw):
    torch, m, oracle_mod, _ = env
    pp = m.FFPP.for_workload(w, **kw)
    out = pp.run(torch.from_numpy(w.raw).cuda(), w.N_per_frame, w.frame_dims)
    torch.cuda.synchronize()
    ref = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
    compare(out, ref, w, check_stage=pp)
    return out, ref


def frame(N, dtype, rng, n_pass, spread=600.0, lo=2.0, hi=6.0):
    """Background frame with n_pass random survivors at random candidates (tie-free unless asked)."""
    raw = np.zeros((N, 5), dtype=dtype)
    raw[:, :4] = 1.0
    raw[:, 4] = -8.0
    if n_pass:
        js = rng.choice(N, size=n_pass, replace=False)
        raw[js, :4] = rng.uniform(0.5, 3.0, size=(n_pass, 4))
        raw[js, 4] = rng.uniform(lo, hi, size=n_pass)
    return raw


@pytest.mark.parametrize("dt", ["fp16", "fp32"])
@pytest.mark.parametrize("n_pass", [0, 1, 2, 63, 64, 65, 127, 128, 129, 1000])
def test_survivor_counts_around_tile_boundaries(env, dt, n_pass):
    rng = np.random.default_rng(100 + n_pass)
    npdt = np.float16 if dt == "fp16" else np.float32
    w = W(frame(8400, npdt, rng, n_pass), [[640, 640]], dict(P, dtype=dt))
    out, ref = check(env, w)
    assert ref.survivor_counts[0] == n_pass


def test_all_pass_none_pass_and_topk_cut(env):
    rng = np.random.default_rng(3)
    raw = frame(8400, np.float16, rng, 0)
    raw[:, 4] = rng.uniform(-1.0, 8.0, size=8400)      # everything above logit(0.25) = -1.0986
    raw[:, :4] = rng.uniform(0.2, 1.5, size=(8400, 4))
    for K in (1, 64, 100, 3000, 8400, 12000):
        w = W(raw, [[640, 640]], dict(P, top_k=K, iou_thresh=0.6))
        out, ref = check(env, w)
        assert ref.survivor_counts[0] == 8400 and ref.sorted_counts[0] == min(K, 8400)
    w = W(frame(8400, np.float16, rng, 0), [[640, 640]], P)
    out, ref = check(env, w)
    assert ref.counts[0] == 0 and not out.density_numpy().any()


def test_equal_scores_and_signed_zero_ties(env):
    rng = np.random.default_rng(4)
    for dt, npdt in (("fp16", np.float16), ("fp32", np.float32)):
        raw = frame(8400, npdt, rng, 0)
        js = rng.choice(8400, size=2000, replace=False)
        vals = np.array([-0.5, 0.0, -0.0, 0.5, 1.0, 2.0, 3.0], dtype=npdt)
        raw[js, 4] = vals[rng.integers(0, len(vals), size=2000)]
        raw[js, :4] = rng.uniform(0.2, 1.0, size=(2000, 4))
        w = W(raw, [[640, 640]], dict(P, dtype=dt, top_k=777, iou_thresh=1.0))
        out, ref = check(env, w)
        assert ref.counts[0] == 777                     # thr >= 1: kept list == sorted top-K list


def test_boxes_outside_the_frame_and_border_cells(env):
    rng = np.random.default_rng(5)
    raw = frame(8400, np.float32, rng, 0)
    # survivors along the frame border with large one-sided distances -> centroids outside / on the border cell
    border = [0, 79, 80 * 79, 6399, 6400, 6439, 8000, 8399, 40, 80 * 40]
    for k, j in enumerate(border):
        raw[j] = [30.0 - 3 * k, 0.5, 0.5 + 3 * k, 0.5, 5.0 - 0.1 * k]
    raw[3000] = [0.5, 40.0, 0.5, 0.25, 6.0]
    raw[3100] = [0.5, 0.25, 0.5, 60.0, 6.5]
    w = W(raw, [[640, 640]], dict(P, dtype="fp32", iou_thresh=0.9))
    out, ref = check(env, w)
    b = ref.boxes[0, :ref.counts[0]]
    cx = (b["x1"] + b["x2"]) / 2
    assert (cx < 0).any() or (cx >= 640).any()          # the case really has out-of-frame centroids


def test_720p_partial_row_and_ragged_mix(env):
    torch, m, oracle_mod, gen = env
    rng = np.random.default_rng(6)
    dims = [[1280, 720], [640, 640], [1280, 720], [1920, 1088], [1280, 720], [64, 64]]
    parts = []
    for W_, H_ in dims:
        N = gen.frame_candidates(W_, H_)
        fr = frame(N, np.float16, rng, min(N // 3, 2500), lo=0.0, hi=8.0)
        fr[N - 20:, 4] = 9.0                           # the half row of 1280x720 (A21) survives
        parts.append(fr)
    w = W(np.concatenate(parts), dims, dict(P, top_k=2000, iou_thresh=0.5, sigma_cells=2.5))
    check(env, w)


def test_many_tiny_frames_take_the_generic_compaction_path(env):
    torch, m, oracle_mod, gen = env
    rng = np.random.default_rng(7)
    dims = [[64, 64]] * 150                              # N = 84 per frame: > 16 frames per 2048-candidate chunk
    parts = [frame(84, np.float16, rng, int(rng.integers(0, 60)), lo=0.0, hi=8.0) for _ in dims]
    w = W(np.concatenate(parts), dims, dict(P, top_k=50, sigma_cells=1.0))
    check(env, w)


@pytest.mark.parametrize("B", [297, 400, 1100])
def test_more_frames_than_resident_ctas(env, B):
    """B above 2 x SM count (a4's CTAs no longer all start at once) and above the 1024-frame limit of the
    weight-ordered CTA -> frame maps of a2 / a4 (identity map)."""
    torch, m, oracle_mod, gen = env
    rng = np.random.default_rng(B)
    dims = [[64, 64] if i % 3 else [128, 64] for i in range(B)]
    parts = [frame(gen.frame_candidates(a, b), np.float16, rng, int(rng.integers(0, 70)), lo=0.0, hi=8.0) for a, b in dims]
    w = W(np.concatenate(parts), dims, dict(P, top_k=40, sigma_cells=1.0))
    check(env, w)


def test_max_topk_for_both_key_widths(env):
    rng = np.random.default_rng(8)
    N = 42840
    raw = frame(N, np.float16, rng, 0)
    raw[:, 4] = rng.uniform(-1.0, 8.0, size=N)
    raw[:, :4] = rng.uniform(0.1, 0.6, size=(N, 4))
    w = W(raw, [[1920, 1088]], dict(P, top_k=24576, iou_thresh=0.7, sigma_cells=3.0))
    check(env, w)
    w32 = W(raw.astype(np.float32), [[1920, 1088]], dict(P, dtype="fp32", top_k=12288, iou_thresh=0.7, sigma_cells=3.0))
    check(env, w32)


def test_keep_everything_at_max_topk_takes_the_global_sort_scratch(env):
    """thr >= 1 keeps the whole top-K list, so the kept set (24576 / 12288 boxes) is far beyond what a4 can order in
    shared memory: the radix passes run on the global scratch arrays."""
    rng = np.random.default_rng(9)
    N = 42840
    raw = frame(N, np.float16, rng, 0)
    raw[:, 4] = rng.uniform(-1.0, 8.0, size=N)
    raw[:, :4] = rng.uniform(0.1, 0.6, size=(N, 4))
    w = W(raw, [[1920, 1088]], dict(P, top_k=24576, iou_thresh=1.0, sigma_cells=2.0))
    out, ref = check(env, w)
    assert ref.counts[0] == 24576
    w32 = W(raw.astype(np.float32), [[1920, 1088]], dict(P, dtype="fp32", top_k=12288, iou_thresh=1.0, sigma_cells=2.0))
    out, ref = check(env, w32)
    assert ref.counts[0] == 12288


@pytest.mark.parametrize("thr", [0.0, 0.02, 0.05, 0.3, 0.5, 0.7, 0.95])
def test_wild_box_sizes_against_every_threshold(env, thr):
    """Boxes from a fraction of a pixel to several frames wide, nested and far outside the frame: the a3 partner window
    (rho * own size around the own centre, in spatial cells) must still reach every pair the oracle's all-pairs walk sees."""
    rng = np.random.default_rng(int(thr * 100) + 11)
    N = 8400
    raw = frame(N, np.float32, rng, 0)
    js = rng.choice(N, size=3000, replace=False)
    raw[js, :4] = np.exp(rng.uniform(np.log(0.02), np.log(60.0), size=(3000, 4))).astype(np.float32)
    big = js[:40]
    raw[big, :4] = rng.uniform(30.0, 120.0, size=(40, 4))            # boxes that cover the whole frame and more
    twins = js[100:400]
    raw[twins, :4] = raw[twins[0], :4] * rng.uniform(0.97, 1.03, size=(300, 4))   # a pile of near-identical shapes
    raw[js, 4] = rng.uniform(-1.0, 8.0, size=3000)
    w = W(raw, [[640, 640]], dict(P, dtype="fp32", top_k=2500, iou_thresh=thr))
    check(env, w)                                        # default pool: whatever does not fit goes through the overflow path
    if thr in (0.0, 0.5):
        check(env, w, nms_edges_per_box=1300)           # and with room for every pair (at thr ~ 0 the frame-sized boxes touch everything)


def test_large_birds_on_the_finest_level_overflow_the_default_pool_and_still_match(env):
    """A bird 120 px wide lights up ~120 stride-8 candidates that all regress (almost) the same box: ~60 suppression pairs
    per box, far beyond the default 16 per top-K slot.  The frame must be bit-exact all the same."""
    torch, m, oracle_mod, gen = env
    rng = np.random.default_rng(21)
    N = 8400
    raw = frame(N, np.float16, rng, 0)
    centres = rng.uniform(90.0, 550.0, size=(24, 2))
    for cx, cy in centres:
        for iy in range(80):
            for ix in range(80):
                px, py = (ix + 0.5) * 8, (iy + 0.5) * 8
                if abs(px - cx) < 44 and abs(py - cy) < 44:
                    j = iy * 80 + ix
                    jit = rng.normal(0.0, 1.5, size=4)
                    raw[j, :4] = (np.array([px - (cx - 60), py - (cy - 60), (cx + 60) - px, (cy + 60) - py]) + jit) / 8.0
                    raw[j, 4] = rng.uniform(1.0, 6.0)
    w = W(raw, [[640, 640]], dict(P, iou_thresh=0.5))
    pp = m.FFPP.for_workload(w)
    out = pp.run(torch.from_numpy(w.raw).cuda(), w.N_per_frame, w.frame_dims)
    torch.cuda.synchronize()
    assert pp.debug_read(5, 1)[0] == 1, "the case is meant to overflow the default pool"
    compare(out, oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims), w, check_stage=pp)


def _iou32(a, b):
    """numpy restatement of O5, op by op in fp32 — only used to CHOOSE cases; the expected result is the oracle's."""
    f = np.float32
    iw = max(f(0), f(min(a[2], b[2]) - max(a[0], b[0])))
    ih = max(f(0), f(min(a[3], b[3]) - max(a[1], b[1])))
    inter = f(iw * ih)
    aa = f(f(a[2] - a[0]) * f(a[3] - a[1]))
    ab = f(f(b[2] - b[0]) * f(b[3] - b[1]))
    return f(inter / f(f(aa + ab) - inter))


@pytest.mark.parametrize("thr", [float(np.float32(1.0) / np.float32(3.0)), 0.45, 0.5, 0.7])
def test_pairs_at_and_around_the_iou_threshold(env, thr):
    """Hand-built pairs whose fp32 IoU equals thr, is one ulp above / below it, and sits just inside / outside the
    2^-20 guard band of iou_exceeds: the exact __fdiv_rn branch decides, as the oracle's division does.  One pair per
    64x64 frame, coordinates below 32 px on a 2^-19 lattice so that one lattice step moves the IoU by ~2 ulps."""
    torch, m, oracle_mod, gen = env
    f32 = np.float32
    t32 = f32(thr)
    rng = np.random.default_rng(int(thr * 1000))
    q = 2.0 ** -19
    pairs = []
    if abs(thr - 0.5) < 1e-9:
        pairs.append((np.array([1, 2, 4, 3], f32), np.array([2, 2, 5, 3], f32)))        # inter 2, union 4: exactly 0.5
    if abs(thr - 1 / 3) < 1e-6:
        pairs.append((np.array([1, 2, 3, 3], f32), np.array([2, 2, 4, 3], f32)))        # inter 1, union 3: fl(1/3)
    for _ in range(40):
        wa, ha = np.round(rng.uniform(9, 14, 2) / q) * q
        wb, hb = np.round(np.array([wa, ha]) * rng.uniform(0.9, 1.1, 2) / q) * q
        A = np.array([2, 2, 2 + wa, 2 + ha], f32)
        lo, hi = 0.0, float(wa)                        # B = A-sized box shifted right by d: IoU falls from ~1 to 0
        for _ in range(60):
            mid = np.round((lo + hi) / 2 / q) * q
            Bx = np.array([2 + mid, 2, 2 + mid + wb, 2 + hb], f32)
            if _iou32(A, Bx) > t32: lo = mid
            else: hi = mid
        for k in range(-6, 7):
            d = lo + k * q
            pairs.append((A, np.array([2 + d, 2, 2 + d + wb, 2 + hb], f32)))
    ious = np.array([_iou32(a, b) for a, b in pairs], f32)
    rel = np.abs(ious.astype(np.float64) - float(t32)) / float(t32)
    assert (rel < 2.0 ** -20).sum() >= 20 and (ious > t32).any() and (ious <= t32).any()
    assert (ious == t32).any() or (np.abs(ious.view(np.int32) - t32.view(np.int32)) <= 1).any(), "no pair within one ulp of thr"
    dims, parts = [], []
    for a, b in pairs:
        fr = np.zeros((84, 5), np.float32); fr[:, :4] = 0.25; fr[:, 4] = -9.0
        # A regressed from candidate (ix=1, iy=1): p = (12, 12); B from (ix=2, iy=1): p = (20, 12); stride 8
        fr[9] = [(12 - a[0]) / 8, (12 - a[1]) / 8, (a[2] - 12) / 8, (a[3] - 12) / 8, 3.0]
        fr[10] = [(20 - b[0]) / 8, (12 - b[1]) / 8, (b[2] - 20) / 8, (b[3] - 12) / 8, 2.0]
        parts.append(fr); dims.append([64, 64])
    w = W(np.concatenate(parts), dims, dict(P, dtype="fp32", iou_thresh=thr, top_k=16, sigma_cells=1.0))
    out, ref = check(env, w)
    dec = out.boxes_numpy()
    for i, (a, b) in enumerate(pairs):                 # the decoded boxes ARE the intended ones, and the decision is the IoU's
        assert np.array_equal(np.array(list(dec[i, 0])[:4], f32), a)
        assert int(ref.counts[i]) == (1 if ious[i] > t32 else 2), (i, ious[i])


def test_output_buffers_at_odd_offsets(env):
    """out_density only needs 4-byte alignment (the float4 store path must look at the pointer, not only
    at the offsets inside the batch); grids of 16-px and 32-px cells give per-frame sizes that are not multiples of 4."""
    torch, m, oracle_mod, gen = env
    rng = np.random.default_rng(31)
    dims = [[160, 96], [224, 96], [640, 640], [160, 96]]
    for cell, sig in ((32, 1.0), (16, 1.0), (8, 2.0)):
        parts = [frame(gen.frame_candidates(a, b), np.float16, rng, 40, lo=0.0, hi=8.0) for a, b in dims]
        w = W(np.concatenate(parts), dims, dict(P, cell_px=cell, sigma_cells=sig, truncate_sigmas=1.0 if cell == 32 else 3.0))
        pp = m.FFPP.for_workload(w)
        ref = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
        for shift in (0, 1, 2, 3):
            out = pp.alloc_outputs(len(dims), w.frame_dims)
            cells = int(out.density_offsets[-1])
            big = torch.full((cells + 8,), -1.0, dtype=torch.float32, device="cuda")
            out.density = big[shift:shift + cells]
            pp.run(torch.from_numpy(w.raw).cuda(), w.N_per_frame, w.frame_dims, out=out)
            torch.cuda.synchronize()
            compare(out, ref, w)
            assert (big[:shift] == -1).all() and (big[shift + cells:] == -1).all()


def test_cuda_graph_capture_and_replay(env):
    """include/ffpp.h: ffpp_run is capturable once the batch geometry is cached.  Capture one run, replay it on
    NEW inputs written into the same buffers, compare with the oracle; an uncached geometry under capture is refused."""
    torch, m, oracle_mod, gen = env
    w0 = gen.make_config(5, B=8, seed_offset=3)
    w1 = gen.make_config(5, B=8, seed_offset=4)
    pp = m.FFPP.for_workload(w0)
    raw = torch.from_numpy(w0.raw).cuda()
    out = pp.alloc_outputs(w0.B, w0.frame_dims)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        pp.run(raw, w0.N_per_frame, w0.frame_dims, out=out)          # caches the geometry
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        pp.run(raw, w0.N_per_frame, w0.frame_dims, out=out)
    out.counts.zero_(); out.density.zero_()
    g.replay(); torch.cuda.synchronize()
    compare(out, oracle_mod.run(w0.params, w0.raw, w0.N_per_frame, w0.frame_dims), w0)
    raw.copy_(torch.from_numpy(w1.raw))
    for _ in range(2):
        g.replay()
    torch.cuda.synchronize()
    compare(out, oracle_mod.run(w1.params, w1.raw, w1.N_per_frame, w1.frame_dims), w1)
    # a geometry the handle has not seen cannot be captured (its descriptor upload reads host memory)
    w2 = gen.make_config(5, B=4, seed_offset=3)
    raw2 = torch.from_numpy(w2.raw).cuda()
    out2 = pp.alloc_outputs(w2.B, w2.frame_dims)
    g2 = torch.cuda.CUDAGraph()
    with pytest.raises(m.FFPPError) as ei:
        with torch.cuda.graph(g2):
            pp.run(raw2, w2.N_per_frame, w2.frame_dims, out=out2)
    assert ei.value.code == m.FFPP_EINVAL and "capture" in str(ei.value)
    torch.cuda.synchronize()


def test_alternating_geometries_never_wait_for_the_device(env):
    """ffpp_run never synchronises the host.  With ~0.3 s of spinning queued ahead on the stream, calls with
    a cached geometry, a NEW geometry and the first one again must all return while the spin is still running."""
    import time
    torch, m, oracle_mod, gen = env
    wa = gen.make_config(5, B=4)
    wb = gen.make_config(5, B=3, seed_offset=1)
    wc = gen.make_config(5, B=6, seed_offset=2)
    big = gen.make_config(5, B=8)
    pp = m.FFPP.for_workload(big)
    ra, rb, rc = (torch.from_numpy(x.raw).cuda() for x in (wa, wb, wc))
    oa = pp.run(ra, wa.N_per_frame, wa.frame_dims)
    torch.cuda.synchronize()
    st = torch.cuda.current_stream()
    torch.cuda._sleep(int(0.3 * 1.9e9))
    t0 = time.perf_counter()
    oa = pp.run(ra, wa.N_per_frame, wa.frame_dims)
    ob = pp.run(rb, wb.N_per_frame, wb.frame_dims)               # new geometry: descriptor build + stream-ordered upload
    oc = pp.run(rc, wc.N_per_frame, wc.frame_dims)               # another new one
    oa2 = pp.run(ra, wa.N_per_frame, wa.frame_dims)
    dt = time.perf_counter() - t0
    still_running = not st.query()
    torch.cuda.synchronize()
    assert still_running and dt < 0.1, f"ffpp_run blocked the host: {dt:.3f} s, spin still running: {still_running}"
    for o, x in ((oa2, wa), (ob, wb), (oc, wc)):
        compare(o, oracle_mod.run(x.params, x.raw, x.N_per_frame, x.frame_dims), x)


@pytest.mark.parametrize("sigma,trunc,R", [(0.5, 3.0, 1), (1.0, 3.0, 3), (1.7, 3.0, 5), (3.7, 3.0, 11), (4.4, 3.0, 13),
                                            (5.8, 3.0, 17), (7.0, 3.0, 21), (10.0, 3.0, 30), (8.0, 4.0, 32)])
def test_every_radius_bucket_of_the_density_kernel(env, sigma, trunc, R):
    """a6 is compiled for a list of radii and runs the smallest one >= R with zero-padded taps."""
    rng = np.random.default_rng(12)
    dims = [[640, 640], [1280, 720], [320, 320]]
    parts = [frame(env[3].frame_candidates(a, b), np.float16, rng, 300, lo=0.0, hi=8.0) for a, b in dims]
    w = W(np.concatenate(parts), dims, dict(P, sigma_cells=sigma, truncate_sigmas=trunc, iou_thresh=0.5))
    torch, m, oracle_mod, _ = env
    assert oracle_mod.taps(sigma, trunc)[0] == R
    check(env, w)


def test_non_finite_inputs_do_not_hang_and_agree_with_the_oracle(env):
    """NaN logits never survive; non-finite distances must not hang or crash (their result is otherwise
    unspecified).  Both sides happen to agree on them too: a box with a NaN/inf coordinate never suppresses and is
    never suppressed (IoU is NaN or 0), and its centroid fails the in-frame test."""
    torch, m, oracle_mod, gen = env
    w = gen.make_config(2, B=2)
    raw = w.raw.copy()
    rng = np.random.default_rng(0)
    js = rng.choice(8400, size=40, replace=False)
    vals = [np.inf, -np.inf, np.nan, 60000.0, -60000.0]
    for k, j in enumerate(js):
        raw[j, k % 4] = vals[k % 5]
        raw[j, 4] = 6.0 - 0.01 * k
    raw[js[0] + 1, 4] = np.nan
    raw[js[1] + 1, 4] = np.inf
    pp = m.FFPP.for_workload(w)
    out = pp.run(torch.from_numpy(raw).cuda(), w.N_per_frame, w.frame_dims)
    torch.cuda.synchronize()
    ref = oracle_mod.run(w.params, raw, w.N_per_frame, w.frame_dims)
    assert np.array_equal(out.counts_numpy(), ref.counts)
    g = out.boxes_numpy()
    for f in range(2):
        n = int(ref.counts[f])
        assert np.array_equal(g[f, :n]["cand_index"], ref.boxes[f, :n]["cand_index"])
        for k in ("x1", "y1", "x2", "y2"):
            a, b = g[f, :n][k], ref.boxes[f, :n][k]
            fin = np.isfinite(b)
            assert np.array_equal(a[fin].view(np.uint32), b[fin].view(np.uint32)) and np.array_equal(np.isnan(a), np.isnan(b))
    d = out.density_numpy()
    assert np.isfinite(d).all() and np.all(np.abs(d - ref.density) <= np.maximum(1e-5, 1e-4 * np.abs(ref.density)))


def test_abi_misuse_is_rejected(env):
    torch, m, oracle_mod, gen = env
    good = dict(max_frames=2, max_total_candidates=2 * 8400, max_frame_w=640, max_frame_h=640)
    for bad in (dict(P, dtype="fp16", top_k=0), dict(P, strides=[8, 24, 32]), dict(P, iou_thresh=-0.1),
                dict(P, sigma_cells=0.0), dict(P, top_k=30000), dict(P, strides=[16, 8, 32])):
        with pytest.raises(m.FFPPError) as ei:
            m.FFPP(bad, **good)
        assert ei.value.code == m.FFPP_EINVAL
    pp = m.FFPP(P, **good)
    raw = torch.zeros((8400, 5), dtype=torch.float16, device="cuda")
    out = pp.alloc_outputs(1, [[640, 640]])
    N = np.array([8400], dtype=np.int32); dims = np.array([[640, 640]], dtype=np.int32)
    args = lambda **k: dict(dict(raw_ptr=raw.data_ptr(), B=1, N_ptr=N.ctypes.data, dims_ptr=dims.ctypes.data, stream_ptr=None,
                                 boxes_ptr=out.boxes.data_ptr(), counts_ptr=out.counts.data_ptr(),
                                 density_ptr=out.density.data_ptr()), **k)
    assert pp.run_raw_pointers(**args()) == m.FFPP_OK
    assert pp.run_raw_pointers(**args(B=0)) == m.FFPP_OK
    assert pp.run_raw_pointers(**args(B=-1)) == m.FFPP_EINVAL
    assert pp.run_raw_pointers(**args(raw_ptr=None)) == m.FFPP_EINVAL
    assert pp.run_raw_pointers(**args(boxes_ptr=None)) == m.FFPP_EINVAL
    assert pp.run_raw_pointers(**args(raw_ptr=raw.data_ptr() + 2)) == m.FFPP_EINVAL and "aligned" in pp.last_error()
    assert pp.run_raw_pointers(**args(B=3)) == m.FFPP_ECAPACITY
    badN = np.array([8399], dtype=np.int32)
    assert pp.run_raw_pointers(**args(N_ptr=badN.ctypes.data)) == m.FFPP_EINVAL
    for d in ([[648, 640]], [[640, 644]], [[1280, 1280]]):
        dd = np.array(d, dtype=np.int32)
        nn = np.array([gen.frame_candidates(*d[0])], dtype=np.int32)
        rc = pp.run_raw_pointers(**args(dims_ptr=dd.ctypes.data, N_ptr=nn.ctypes.data))
        assert rc in (m.FFPP_EINVAL, m.FFPP_ECAPACITY) and rc != m.FFPP_OK
    torch.cuda.synchronize()
    pp.close()
