"""Pins for the CPU oracle (oracle/ffpp_oracle.cpp): hand-worked cases, closed forms, invariants,
brute force and reductions to library routines — nothing here re-types the oracle's own code path.

Sources: BASELINE.json north_star (hand cases it demands), SURVEY.md §8(c) "Pins", tests/golden/*.txt.
"""
import math

import numpy as np
import pytest

from conftest import golden_rows

P640 = dict(dtype="fp32", conf_thresh=0.25, iou_thresh=0.45, top_k=3000, strides=[8, 16, 32], cell_px=8,
            sigma_cells=2.0, truncate_sigmas=3.0)
N640 = 8400


def background(N, dtype=np.float32, logit=-10.0):
    """A frame in which nothing passes the threshold: unit distances, logit far below any T."""
    raw = np.zeros((N, 5), dtype=dtype)
    raw[:, :4] = 1.0
    raw[:, 4] = logit
    return raw


# ------------------------------------------------------------------ half conversion (library reduction: numpy)
def test_half_to_float_matches_numpy_for_all_bit_patterns(oracle_mod):
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float32)
    got = np.array([oracle_mod.half_to_float(int(b)) for b in bits], dtype=np.float32)
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan].view(np.uint32), ref[~nan].view(np.uint32))


# ------------------------------------------------------------------ O3 threshold closed form
def test_logit_threshold_closed_forms(oracle_mod):
    for conf, val in golden_rows("logit_thresholds.txt"):
        got = oracle_mod.logit_threshold(float(conf))
        assert got == np.float32(float(val)), (conf, got)
    assert oracle_mod.logit_threshold(0.0) == -math.inf
    assert oracle_mod.logit_threshold(1.0) == math.inf


def test_threshold_is_strict_and_one_ulp_flips_membership(oracle_mod):
    T = np.float32(oracle_mod.logit_threshold(0.25))
    raw = background(N640)
    raw[10, 4] = T                                   # equal -> not a survivor (strict >)
    raw[20, 4] = np.nextafter(T, np.float32(np.inf))  # one ulp above -> survivor
    raw[30, 4] = np.nextafter(T, np.float32(-np.inf))
    raw[40, 4] = np.nan                              # NaN fails the comparison (A6)
    r = oracle_mod.run(P640, raw, [N640], [[640, 640]])
    assert r.survivor_counts[0] == 1
    assert r.counts[0] == 1 and r.boxes[0, 0]["cand_index"] == 20
    # fp16 rows: threshold compared after exact widening to fp32
    p = dict(P640, dtype="fp16")
    rawh = background(N640, np.float16)
    below = np.float16(T)                            # RNE of T; find the fp16 neighbours around T
    lo = below if np.float32(below) <= T else np.nextafter(below, np.float16(-np.inf))
    hi = np.nextafter(lo, np.float16(np.inf))
    assert np.float32(lo) <= T < np.float32(hi)
    rawh[5, 4], rawh[6, 4] = lo, hi
    r = oracle_mod.run(p, rawh, [N640], [[640, 640]])
    assert r.survivor_counts[0] == 1 and r.boxes[0, 0]["cand_index"] == 6


# ------------------------------------------------------------------ O1/O2 decode hand cases (D1)
def test_decode_hand_cases(oracle_mod):
    for row in golden_rows("decode_hand_cases.txt"):
        j = int(row[0]); ltrb = [float(x) for x in row[1:5]]
        loc = tuple(int(x) for x in row[5:8]); box = [float(x) for x in row[8:12]]
        got, gloc = oracle_mod.decode_candidate(P640, 640, 640, j, ltrb)
        assert gloc == loc, (j, gloc)
        assert got.tolist() == box, (j, got)


def test_decode_hand_cases_through_the_whole_path_fp32_and_fp16(oracle_mod):
    for dt, npdt in (("fp32", np.float32), ("fp16", np.float16)):
        raw = background(N640, npdt)
        rows = golden_rows("decode_hand_cases.txt")
        expect = {}
        for k, row in enumerate(rows):
            j = int(row[0])
            if j in expect:
                continue
            raw[j, :4] = [float(x) for x in row[1:5]]
            raw[j, 4] = 5.0 - k                     # distinct scores
            expect[j] = [float(x) for x in row[8:12]]
        # thr >= 1: NMS keeps everything (IoU <= 1 is never > 1)
        r = oracle_mod.run(dict(P640, dtype=dt, iou_thresh=1.0), raw, [N640], [[640, 640]])
        assert r.counts[0] == len(expect)
        for b in r.boxes[0, :r.counts[0]]:
            assert [b["x1"], b["y1"], b["x2"], b["y2"]] == expect[int(b["cand_index"])]


def test_720p_partial_row_layout(oracle_mod, gen_mod):
    # A21: 1280x720 -> 14400 + 3600 + 900 = 18900; stride-32 level has 22 full rows + 20 candidates with py = 720
    assert gen_mod.frame_candidates(1280, 720) == 18900
    j = 14400 + 3600 + 880 + 7
    got, loc = oracle_mod.decode_candidate(P640, 1280, 720, j, [0, 0, 0, 0])
    assert loc == (32, 7, 22) and got.tolist() == [240.0, 720.0, 240.0, 720.0]
    got, loc = oracle_mod.decode_candidate(P640, 1280, 720, 18899, [0, 0, 0, 0])
    assert loc == (32, 19, 22)
    got, loc = oracle_mod.decode_candidate(P640, 1280, 720, 14400, [0, 0, 0, 0])
    assert loc == (16, 0, 0) and got.tolist() == [8.0, 8.0, 8.0, 8.0]


# ------------------------------------------------------------------ O5 IoU hand case (N1)
def test_two_box_iou_just_above_and_below_threshold(oracle_mod):
    for row in golden_rows("nms_two_box_case.txt"):
        ja, la, ta, ra, ba, za = int(row[1]), *[float(x) for x in row[2:7]]
        jb, lb, tb, rb, bb, zb = int(row[7]), *[float(x) for x in row[8:13]]
        num, den = int(row[13]), int(row[14])
        kept = [int(x) for x in row[15].split(",")]
        boxa, _ = oracle_mod.decode_candidate(P640, 640, 640, ja, [la, ta, ra, ba])
        boxb, _ = oracle_mod.decode_candidate(P640, 640, 640, jb, [lb, tb, rb, bb])
        got = oracle_mod.iou(boxa, boxb)
        assert got == np.float32(num) / np.float32(den)          # 6300/13700 reduces exactly
        assert got == oracle_mod.iou(boxb, boxa)                  # symmetric
        for dt, npdt in (("fp32", np.float32), ("fp16", np.float16)):
            raw = background(N640, npdt)
            raw[ja] = [la, ta, ra, ba, za]
            raw[jb] = [lb, tb, rb, bb, zb]
            r = oracle_mod.run(dict(P640, dtype=dt), raw, [N640], [[640, 640]])
            assert r.boxes[0, :r.counts[0]]["cand_index"].tolist() == kept, row[0]


def test_iou_textbook_cases(oracle_mod):
    a = [0, 0, 10, 10]
    assert oracle_mod.iou(a, a) == 1.0
    assert oracle_mod.iou(a, [10, 0, 20, 10]) == 0.0            # touching edges: zero intersection
    assert oracle_mod.iou(a, [20, 20, 30, 30]) == 0.0
    assert oracle_mod.iou(a, [5, 0, 15, 10]) == np.float32(50) / np.float32(150)
    assert oracle_mod.iou(a, [2, 2, 8, 8]) == np.float32(36) / np.float32(100)   # containment
    assert math.isnan(oracle_mod.iou([1, 1, 1, 1], [1, 1, 1, 1]))                 # 0/0, A12: never suppresses
    assert list(oracle_mod.nms_sorted([[1, 1, 1, 1], [1, 1, 1, 1]], 0.0)) == [0, 1]
    # strict >: IoU exactly equal to the threshold does not suppress (A11)
    assert list(oracle_mod.nms_sorted([a, [5, 0, 15, 10]], float(np.float32(50) / np.float32(150)))) == [0, 1]
    assert list(oracle_mod.nms_sorted([a, [5, 0, 15, 10]], 0.33)) == [0]


def test_iou_exactly_at_threshold_does_not_suppress_in_the_whole_path(oracle_mod):
    # A11 strict >.  A = (2,2,102,102); B = A shifted 50 px down: inter 5000, union 15000, IoU = fl(1/3) exactly.
    thr = float(np.float32(1) / np.float32(3))
    raw = background(N640)
    raw[486] = [6.25, 6.25, 6.25, 6.25, 2.0]
    raw[966] = [6.25, 6.0, 6.25, 6.5, 1.0]          # cell (6,12): p = (52,100) -> (2,52,102,152)
    r = oracle_mod.run(dict(P640, iou_thresh=thr), raw, [N640], [[640, 640]])
    assert r.boxes[0, :r.counts[0]]["cand_index"].tolist() == [486, 966]
    b = r.boxes[0, 1]
    assert [b["x1"], b["y1"], b["x2"], b["y2"]] == [2.0, 52.0, 102.0, 152.0]
    below = float(np.nextafter(np.float32(thr), np.float32(0)))
    r = oracle_mod.run(dict(P640, iou_thresh=below), raw, [N640], [[640, 640]])
    assert r.boxes[0, :r.counts[0]]["cand_index"].tolist() == [486]


# ------------------------------------------------------------------ O5 brute force + library reduction
def random_boxes(rng, n, extent=100.0, size=30.0):
    c = rng.uniform(0, extent, size=(n, 2))
    wh = rng.uniform(0.3 * size, size, size=(n, 2))
    return np.concatenate([c - wh / 2, c + wh / 2], axis=1).astype(np.float32)


def brute_force_nms(boxes, thr):
    """Full O(n^2) IoU matrix in numpy fp32 (op by op), then the greedy sweep over the matrix."""
    b = boxes.astype(np.float32)
    x1, y1, x2, y2 = b[:, 0], b[:, 1], b[:, 2], b[:, 3]
    iw = np.maximum(np.float32(0), np.minimum(x2[:, None], x2[None, :]) - np.maximum(x1[:, None], x1[None, :]))
    ih = np.maximum(np.float32(0), np.minimum(y2[:, None], y2[None, :]) - np.maximum(y1[:, None], y1[None, :]))
    inter = iw * ih
    area = (x2 - x1) * (y2 - y1)
    with np.errstate(invalid="ignore", divide="ignore"):
        M = inter / ((area[:, None] + area[None, :]) - inter)
    assert M.dtype == np.float32
    removed = np.zeros(len(b), bool)
    keep = []
    for i in range(len(b)):
        if removed[i]:
            continue
        keep.append(i)
        removed |= M[i] > np.float32(thr)
        removed[: i + 1] = removed[: i + 1]  # earlier entries irrelevant
    return keep, M


@pytest.mark.parametrize("seed", range(8))
def test_nms_equals_brute_force_on_50_random_boxes(oracle_mod, seed):
    rng = np.random.default_rng(1000 + seed)
    boxes = random_boxes(rng, 50)
    for thr in (0.3, 0.45, 0.5):
        keep, M = brute_force_nms(boxes, thr)
        off = M[np.triu_indices(50, 1)]
        assert np.all(np.abs(off - thr) > 1e-5)
        assert oracle_mod.nms_sorted(boxes, thr).tolist() == keep
        # oracle IoU is the same fp32 value as the numpy op-by-op matrix
        for i, j in [(0, 1), (3, 17), (20, 49)]:
            got = oracle_mod.iou(boxes[i], boxes[j])
            assert got == M[i, j] or (math.isnan(got) and math.isnan(M[i, j]))


@pytest.mark.parametrize("seed", range(4))
def test_nms_equals_torchvision_on_tie_free_inputs(oracle_mod, seed):
    torch = pytest.importorskip("torch")
    tv = pytest.importorskip("torchvision")
    rng = np.random.default_rng(2000 + seed)
    boxes = random_boxes(rng, 300, extent=200.0)
    scores = rng.permutation(300).astype(np.float32)             # distinct -> no tie order question
    order = np.argsort(-scores, kind="stable")
    for thr in (0.45, 0.5):
        ref = tv.ops.nms(torch.from_numpy(boxes), torch.from_numpy(scores), thr).numpy()
        got = order[oracle_mod.nms_sorted(boxes[order], thr)]
        assert got.tolist() == ref.tolist()


def test_nms_invariants_on_a_generated_frame(oracle_mod, gen_mod):
    w = gen_mod.make_config(2, B=2)
    r = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
    thr = np.float32(w.params["iou_thresh"])
    off = 0
    for f in range(w.B):
        n, ns = int(r.counts[f]), int(r.sorted_counts[f])
        assert 0 < n <= ns <= w.params["top_k"]
        kb = np.stack([r.boxes[f, :n][k] for k in ("x1", "y1", "x2", "y2")], axis=1)
        _, M = brute_force_nms(kb, thr)
        assert not np.any(np.triu(M, 1) > thr)                   # no two kept boxes overlap above thr
        # every removed box of the sorted list has IoU > thr with an earlier kept box
        kept_idx = r.boxes[f, :n]["cand_index"]
        sidx = r.sorted_idx[f, :ns]
        kept_pos = {int(c): k for k, c in enumerate(kept_idx)}
        raw = w.raw[off:off + w.N_per_frame[f]].astype(np.float32)
        checked = 0
        for pos, c in enumerate(sidx):
            if int(c) in kept_pos:
                continue
            box, _ = oracle_mod.decode_candidate(w.params, *w.frame_dims[f], int(c), raw[c, :4])
            earlier = [k for k, cc in enumerate(kept_idx) if np.where(sidx == cc)[0][0] < pos]
            assert any(oracle_mod.iou(kb[k], box) > thr for k in earlier)
            checked += 1
            if checked >= 150:
                break
        off += w.N_per_frame[f]


# ------------------------------------------------------------------ O4 sort / top-K (python sorted as the library routine)
def test_sort_order_ties_and_topk_cut(oracle_mod):
    rng = np.random.default_rng(7)
    for dt, npdt in (("fp32", np.float32), ("fp16", np.float16)):
        raw = background(N640, npdt)
        # 500 survivors drawn from only 16 distinct logits -> large equal-score blocks; include +-0 block (A9)
        vals = np.array([-0.5, -0.25, 0.0, -0.0, 0.25, 0.5, 1, 1.5, 2, 2.5, 3, 4, 5, 6, 7, 8], dtype=npdt)
        js = rng.choice(N640, size=500, replace=False)
        raw[js, 4] = vals[rng.integers(0, len(vals), size=500)]
        K = 123
        p = dict(P640, dtype=dt, iou_thresh=1.0, top_k=K)          # thr >= 1: kept list = sorted top-K list
        r = oracle_mod.run(p, raw, [N640], [[640, 640]])
        z = raw[:, 4].astype(np.float32)
        T = np.float32(oracle_mod.logit_threshold(0.25))
        surv = [j for j in range(N640) if z[j] > T]
        expect = sorted(surv, key=lambda j: (-float(z[j]), j))      # -0.0 == 0.0 under float comparison
        assert r.survivor_counts[0] == len(surv) == 500
        assert r.sorted_counts[0] == K
        assert r.sorted_idx[0, :K].tolist() == expect[:K]
        assert r.boxes[0, :r.counts[0]]["cand_index"].tolist() == expect[:K]
        # n < K: nothing cut, padding untouched
        r2 = oracle_mod.run(dict(p, top_k=3000), raw, [N640], [[640, 640]])
        assert r2.sorted_counts[0] == 500 and r2.sorted_idx[0, :500].tolist() == expect
        assert np.all(r2.sorted_idx[0, 500:] == -1)


def test_reported_score_is_sigmoid(oracle_mod):
    raw = background(N640)
    raw[100, 4], raw[200, 4] = 2.0, -1.0
    r = oracle_mod.run(dict(P640, iou_thresh=1.0), raw, [N640], [[640, 640]])
    assert abs(r.boxes[0, 0]["score"] - 1 / (1 + math.exp(-2.0))) < 1e-6
    assert abs(r.boxes[0, 1]["score"] - 1 / (1 + math.exp(1.0))) < 1e-6


# ------------------------------------------------------------------ O7 density (G1 closed form, invariants, scipy)
def gaussian_rows():
    rows = golden_rows("gaussian_constants.txt")
    consts = [(float(r[0]), int(r[1]), float(r[2]), float(r[3])) for r in rows if len(r) == 4]
    named = {r[0]: float(r[1]) for r in rows if len(r) == 2}
    return consts, named


def test_taps_match_printed_constants(oracle_mod):
    consts, named = gaussian_rows()
    for sigma, R, Z, w0 in consts:
        gR, w = oracle_mod.taps(sigma, 3.0)
        assert gR == R and len(w) == 2 * R + 1
        assert abs(w[R] - w0) < 1e-11 and abs(1.0 / w[R] - Z) < 1e-10
        assert abs(w.sum() - 1.0) < 1e-15 and np.array_equal(w, w[::-1])
        for k in range(-R, R + 1):
            assert abs(w[k + R] - math.exp(-k * k / (2 * sigma * sigma)) / Z) < 1e-12
    _, w = oracle_mod.taps(2.0, 3.0)
    assert abs(w[0] - named["w6_sigma2"]) < 1e-9


def test_single_centroid_at_grid_centre_closed_form(oracle_mod):
    consts, named = gaussian_rows()
    Z = consts[0][2]
    D, n_in = oracle_mod.density([[304, 314, 344, 334]], 640, 640, 8, 2.0)   # centre (324,324) -> cell (40,40)
    assert n_in == 1 and D.shape == (80, 80)
    assert abs(D[40, 40] - named["peak_sigma2"]) < 1e-9
    for dy in range(-40, 40):
        for dx in range(-40, 40):
            v = D[40 + dy, 40 + dx]
            if max(abs(dx), abs(dy)) > 6:
                assert v == 0.0
            else:
                assert abs(v - math.exp(-(dx * dx + dy * dy) / 8.0) / (Z * Z)) < 1e-9
    assert abs(float(D.astype(np.float64).sum()) - 1.0) < 1e-6
    # the same through the whole path: one survivor whose box is centred at (324,324)
    raw = background(N640)
    j = 40 * 80 + 40                                 # level 0 cell (40,40): p = (324,324)
    raw[j] = [2.5, 1.25, 2.5, 1.25, 3.0]
    r = oracle_mod.run(P640, raw, [N640], [[640, 640]])
    assert r.counts[0] == 1 and np.array_equal(r.density.reshape(80, 80), D)


def test_density_corner_fold_conserves_mass_and_is_symmetric(oracle_mod):
    D, n_in = oracle_mod.density([[0, 0, 6, 6]], 640, 640, 8, 2.0)          # centroid (3,3) -> cell (0,0)
    assert n_in == 1
    assert abs(float(D.astype(np.float64).sum()) - 1.0) < 1e-6
    assert np.allclose(D, D.T, atol=0, rtol=0)
    _, w = oracle_mod.taps(2.0)
    # 1-D folded profile: cell i gets w[i] + w[-i-1]  (taps index k+R)
    R = 6
    prof = np.array([w[R + i] + (w[R - i - 1] if i + 1 <= R else 0.0) for i in range(R + 1)])
    assert np.allclose(D[0, : R + 1], prof[0] * prof, atol=1e-9)
    assert np.all(D[R + 1:, :] == 0) and np.all(D[:, R + 1:] == 0)
    assert [oracle_mod.fold(i, 5) for i in (-3, -1, 0, 4, 5, 7)] == [2, 0, 0, 4, 4, 2]


def test_density_in_frame_rule_and_counts(oracle_mod):
    # centroids: inside, exactly on the right border (x = W -> out), negative (out), on 0 (in)
    boxes = [[100, 100, 120, 120], [630, 10, 650, 30], [-30, 50, 10, 70], [-10, 40, 10, 60]]
    D, n_in = oracle_mod.density(boxes, 640, 640, 8, 2.0)
    assert n_in == 2
    assert abs(float(D.astype(np.float64).sum()) - 2.0) < 2e-4
    D0, n0 = oracle_mod.density(np.zeros((0, 4), np.float32), 640, 640, 8, 2.0)
    assert n0 == 0 and not D0.any()


@pytest.mark.parametrize("W,H,sigma", [(640, 640, 2.0), (1280, 720, 2.5), (1920, 1088, 3.0)])
def test_density_equals_scipy_reflect_correlation_and_marginals(oracle_mod, W, H, sigma):
    ndi = pytest.importorskip("scipy.ndimage")
    rng = np.random.default_rng(5)
    n = 400
    c = np.stack([rng.uniform(-20, W + 20, n), rng.uniform(-20, H + 20, n)], axis=1)
    c[:40] = np.stack([rng.uniform(0, 30, 40), rng.uniform(0, H, 40)], axis=1)          # crowd the left border
    c[40:60] = [W - 1.0, H - 1.0]                                                      # pile-up in the last cell
    wh = rng.uniform(8, 40, size=(n, 2))
    boxes = np.concatenate([c - wh / 2, c + wh / 2], axis=1).astype(np.float32)
    D, n_in = oracle_mod.density(boxes, W, H, 8, sigma)
    cx = (boxes[:, 0] + boxes[:, 2]) * np.float32(0.5)
    cy = (boxes[:, 1] + boxes[:, 3]) * np.float32(0.5)
    ok = (cx >= 0) & (cx < W) & (cy >= 0) & (cy < H)
    assert n_in == int(ok.sum())
    gw, gh = W // 8, H // 8
    hist = np.zeros((gh, gw))
    np.add.at(hist, (np.floor(cy[ok] / 8).astype(int), np.floor(cx[ok] / 8).astype(int)), 1.0)
    R, w = oracle_mod.taps(sigma)
    ref = ndi.correlate1d(ndi.correlate1d(hist, w, axis=1, mode="reflect"), w, axis=0, mode="reflect")
    assert np.all(np.abs(D - ref) <= np.maximum(1e-6, 1e-6 * np.abs(ref)))
    # invariant (BASELINE.json): grid sums to the in-frame kept count within 1e-4 relative
    assert abs(float(D.astype(np.float64).sum()) - n_in) <= 1e-4 * n_in
    # marginal: column sums = 1-D reflect-convolved column histogram
    assert np.allclose(D.astype(np.float64).sum(axis=0), ndi.correlate1d(hist.sum(axis=0), w, mode="reflect"), atol=1e-4)


# ------------------------------------------------------------------ whole-path properties
def test_frame_independence_and_determinism(oracle_mod, gen_mod):
    w = gen_mod.make_config(2, B=3)
    r = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
    r_again = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
    assert r.boxes.tobytes() == r_again.boxes.tobytes() and r.density.tobytes() == r_again.density.tobytes()
    perm = [2, 0, 1]
    N = int(w.N_per_frame[0])
    raw_p = np.concatenate([w.raw[p * N:(p + 1) * N] for p in perm])
    rp = oracle_mod.run(w.params, raw_p, w.N_per_frame, w.frame_dims)
    for k, p in enumerate(perm):
        assert rp.counts[k] == r.counts[p]
        assert rp.boxes[k].tobytes() == r.boxes[p].tobytes()
        assert np.array_equal(rp.density[6400 * k:6400 * (k + 1)], r.density[6400 * p:6400 * (p + 1)])
    # grid-sum invariant on a real workload
    for f in range(w.B):
        b = r.boxes[f, :r.counts[f]]
        cx = (b["x1"] + b["x2"]) * np.float32(0.5); cy = (b["y1"] + b["y2"]) * np.float32(0.5)
        n_in = int(((cx >= 0) & (cx < 640) & (cy >= 0) & (cy < 640)).sum())
        s = float(r.density[6400 * f:6400 * (f + 1)].astype(np.float64).sum())
        assert abs(s - n_in) <= 1e-4 * max(n_in, 1)


def test_empty_batch_and_empty_frame(oracle_mod):
    r = oracle_mod.run(P640, np.zeros((0, 5), np.float32), [], np.zeros((0, 2), np.int32))
    assert r.counts.shape == (0,)
    r = oracle_mod.run(P640, background(N640), [N640], [[640, 640]])
    assert r.counts[0] == 0 and r.survivor_counts[0] == 0 and not r.density.any()


def test_ragged_batch_equals_each_frame_run_alone(oracle_mod, gen_mod):
    # config 5 layout (A22/A23): mixed resolutions tightly concatenated; per-frame results do not depend on the batch
    w = gen_mod.make_config(5, B=4)
    assert w.frame_dims.tolist() == [[640, 640], [1280, 1280], [1920, 1088], [1280, 720]]
    r = oracle_mod.run(w.params, w.raw, w.N_per_frame, w.frame_dims)
    off = np.concatenate([[0], np.cumsum(w.N_per_frame)])
    assert r.density_offsets.tolist() == [0, 6400, 6400 + 25600, 6400 + 25600 + 32640, 6400 + 25600 + 32640 + 14400]
    for f in range(4):
        one = oracle_mod.run(w.params, w.raw[off[f]:off[f + 1]], w.N_per_frame[f:f + 1], w.frame_dims[f:f + 1])
        assert one.counts[0] == r.counts[f] and one.boxes[0].tobytes() == r.boxes[f].tobytes()
        assert np.array_equal(one.density, r.density[r.density_offsets[f]:r.density_offsets[f + 1]])
        assert one.density.any()
