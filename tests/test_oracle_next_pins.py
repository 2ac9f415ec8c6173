"""Pins of oracle/ffpp_next_oracle.cpp against what the mathematics and library routines fix.
The paper prints no formula or value for any of these steps, so the pins are closed forms,
hand-worked grids, library reductions (scipy.ndimage.label, torch interpolate) and brute force — each chosen so that a
plausible slip (wrong log base, missing normalisation, 8- for 4-connectivity, off-by-one bbox, align_corners) fails one."""
import math

import numpy as np
import pytest

import oracle


# ---------------------------------------------------------------- f1: entropy / clustering degree (B1, B2)
def test_entropy_uniform_grid_is_ln_n():
    for shape in [(1, 2), (4, 4), (80, 80), (136, 240)]:
        n = shape[0] * shape[1]
        for scale in (1.0, 0.037, 123.0):                     # normalisation: scale-free
            D = np.full(shape, scale, dtype=np.float32)
            assert oracle.entropy(D) == pytest.approx(math.log(n), rel=1e-12)
            assert oracle.clustering_degree(D) == pytest.approx(0.0, abs=1e-12)


def test_entropy_single_cell_is_zero_and_degree_one():
    D = np.zeros((9, 7), dtype=np.float32)
    D[3, 5] = 2.5
    assert oracle.entropy(D) == 0.0
    assert oracle.clustering_degree(D) == 1.0


def test_entropy_two_block_grid_by_hand():
    # half the cells hold mass 3 each, the other half mass 1 each: p = 3/(4m) and 1/(4m) with m = n/2 cells each
    D = np.ones((6, 10), dtype=np.float32)
    D[:3] = 3.0
    m = 30
    H = -(m * (3 / (4 * m)) * math.log(3 / (4 * m)) + m * (1 / (4 * m)) * math.log(1 / (4 * m)))
    assert oracle.entropy(D) == pytest.approx(H, rel=1e-12)
    assert oracle.clustering_degree(D) == pytest.approx(1 - H / math.log(60), rel=1e-12)
    # textbook value: two cells 1/4, 3/4 -> 0.5623351446 nats
    assert oracle.entropy(np.array([[1.0, 3.0]], dtype=np.float32)) == pytest.approx(0.5623351446188083, rel=1e-12)


def test_entropy_empty_and_nonpositive_cells():
    assert oracle.entropy(np.zeros((5, 5), dtype=np.float32)) == 0.0
    assert oracle.clustering_degree(np.zeros((5, 5), dtype=np.float32)) == 0.0
    D = np.array([[0.0, 1.0, 1.0, 0.0]], dtype=np.float32)       # zero cells contribute nothing: ln 2
    assert oracle.entropy(D) == pytest.approx(math.log(2), rel=1e-12)
    assert oracle.clustering_degree(D) == pytest.approx(1 - math.log(2) / math.log(4), rel=1e-12)


def test_entropy_against_scipy_on_random_grids():
    from scipy.stats import entropy as sp_entropy
    rng = np.random.default_rng(5)
    for _ in range(5):
        D = rng.gamma(0.3, 1.0, (40, 33)).astype(np.float32)
        D[rng.random(D.shape) < 0.5] = 0
        assert oracle.entropy(D) == pytest.approx(float(sp_entropy(D.astype(np.float64).ravel())), rel=1e-10)


# ---------------------------------------------------------------- f1 / f3: connected components (B3, B5)
def test_regions_hand_case_u_shape_and_diagonal():
    #   a U (one 4-connected region whose two arms meet only at the bottom: the scan meets them as two runs first),
    #   a cell touching it only diagonally (separate under 4-, merged under 8-connectivity), and a lone cell
    g = np.array([[1, 0, 1, 0, 0, 0],
                  [1, 0, 1, 0, 0, 1],
                  [1, 1, 1, 0, 0, 0],
                  [0, 0, 0, 1, 0, 0]], dtype=np.float32) * 2.0
    lab, tab, n = oracle.regions(g, 1.0, conn=4)
    assert n == 3
    assert tab["label"].tolist() == [0, 11, 21]              # smallest row-major index of each region, ascending
    assert tab["area"].tolist() == [7, 1, 1]
    assert (tab["x0"][0], tab["y0"][0], tab["x1"][0], tab["y1"][0]) == (0, 0, 2, 2)
    assert tab["mass"].tolist() == [14.0, 2.0, 2.0]
    assert lab[0, 2] == 0 and lab[2, 1] == 0 and lab[3, 3] == 21 and lab[0, 1] == -1
    lab8, tab8, n8 = oracle.regions(g, 1.0, conn=8)
    assert n8 == 2 and tab8["area"].tolist() == [8, 1] and lab8[3, 3] == 0
    assert (tab8["x1"][0], tab8["y1"][0]) == (3, 3)
    # strict threshold: cells equal to the threshold are background
    assert oracle.regions(g, 2.0, conn=4)[2] == 0


@pytest.mark.parametrize("conn", [4, 8])
def test_regions_against_scipy_label(conn):
    from scipy import ndimage
    rng = np.random.default_rng(11 + conn)
    st = ndimage.generate_binary_structure(2, 1 if conn == 4 else 2)
    for p in (0.35, 0.55, 0.62):                             # around the percolation threshold: large winding components
        D = rng.random((37, 53)).astype(np.float32)
        thr = np.float32(1 - p)
        lab, tab, n = oracle.regions(D, float(thr), conn=conn, max_regions=4096)
        ref, nref = ndimage.label(D > thr, structure=st)
        assert n == nref
        # same partition, and the label is the smallest index of its component
        flat, rflat = lab.ravel(), ref.ravel()
        for k in range(1, nref + 1):
            idx = np.flatnonzero(rflat == k)
            assert (flat[idx] == idx.min()).all()
        assert (flat[rflat == 0] == -1).all()
        areas = ndimage.sum_labels(np.ones_like(D), ref, index=np.arange(1, nref + 1))
        order = np.argsort([np.flatnonzero(rflat == k).min() for k in range(1, nref + 1)])
        assert tab["area"].tolist() == areas[order].astype(int).tolist()
        masses = ndimage.sum_labels(D.astype(np.float64), ref, index=np.arange(1, nref + 1))[order]
        np.testing.assert_allclose(tab["mass"], masses, rtol=1e-6)
        sl = ndimage.find_objects(ref)
        for j, k in enumerate(order):
            ys, xs = sl[k]
            assert (tab["x0"][j], tab["y0"][j], tab["x1"][j], tab["y1"][j]) == (xs.start, ys.start, xs.stop - 1, ys.stop - 1)


def test_regions_table_overflow_reports_total():
    D = np.zeros((8, 8), dtype=np.float32)
    D[::2, ::2] = 1.0                                        # 16 isolated cells
    lab, tab, n = oracle.regions(D, 0.5, conn=4, max_regions=5)
    assert n == 16 and len(tab) == 5 and tab["label"].tolist() == [0, 2, 4, 6, 16]


def test_mask_components_score_min_area_and_fp16():
    m = np.zeros((6, 8), dtype=np.float16)
    m[1:3, 1:4] = np.float16(0.75)                           # 6 pixels
    m[2, 4] = np.float16(0.5)                                # threshold itself: background (strict)
    m[4, 6] = np.float16(0.9)                                # 1 pixel
    m[5, 7] = np.float16(0.625)                              # diagonal neighbour: same component under 8-connectivity
    lab, tab, n = oracle.mask_components(m, 0.5, conn=8, min_area=1)
    assert n == 2 and tab["area"].tolist() == [6, 2]
    assert tab["mass"][0] == np.float32(0.75)
    assert tab["mass"][1] == pytest.approx((float(np.float16(0.9)) + 0.625) / 2, rel=1e-6)
    assert (tab["x0"][1], tab["y0"][1], tab["x1"][1], tab["y1"][1]) == (6, 4, 7, 5)
    lab4, tab4, n4 = oracle.mask_components(m, 0.5, conn=4, min_area=1)
    assert n4 == 3
    lab2, tab2, n2 = oracle.mask_components(m, 0.5, conn=8, min_area=3)
    assert n2 == 1 and tab2["label"].tolist() == [9]        # the small component is left out of the table, not of the labels
    assert lab2[4, 6] == 4 * 8 + 6


def test_mask_components_against_scipy_on_blob_masks():
    from scipy import ndimage
    import flockgen
    masks = flockgen.make_mask_batch(2, 320, 192, birds=60, seed=3)
    for m in masks:
        lab, tab, n = oracle.mask_components(m, 0.5, conn=8)
        ref, nref = ndimage.label(m.astype(np.float32) > 0.5, structure=np.ones((3, 3)))
        assert n == nref and n > 20
        idx_min = ndimage.minimum(np.arange(m.size).reshape(m.shape), ref, index=np.arange(1, nref + 1)).astype(int)
        assert sorted(tab["label"].tolist()) == sorted(idx_min.tolist())
        means = ndimage.mean(m.astype(np.float64), ref, index=np.arange(1, nref + 1))
        np.testing.assert_allclose(tab["mass"], means[np.argsort(idx_min)], rtol=1e-6)


# ---------------------------------------------------------------- f2: exact-position density (B4)
def test_density_exact_centroid_on_cell_centre_reproduces_g1():
    # one box centred (324, 324) -> cell (40, 40) of 80x80, sigma 2, R 6 (tests/golden/density_g1_constants.txt)
    Z, w0 = 5.008122486108, 0.199675627498
    D, n_in = oracle.density_exact([[304, 304, 344, 344]], 640, 640, 8, 2.0)
    assert n_in == 1
    for dy in range(-8, 9):
        for dx in range(-8, 9):
            want = math.exp(-(dx * dx + dy * dy) / 8.0) / (Z * Z) if max(abs(dx), abs(dy)) <= 6 else 0.0
            assert D[40 + dy, 40 + dx] == pytest.approx(want, rel=2e-6, abs=1e-12)
    assert D[40, 40] == pytest.approx(w0 * w0, rel=2e-6)
    assert float(D.sum()) == pytest.approx(1.0, rel=1e-5)
    # and equals the binned oracle there
    Db, _ = oracle.density([[304, 304, 344, 344]], 640, 640, 8, 2.0)
    np.testing.assert_allclose(D, Db, rtol=2e-6, atol=1e-9)


def test_density_exact_off_centre_shifts_the_kernel():
    # centroid at (322, 326): u = 40.25, v = 40.75 -> dx = ix + .5 - 40.25, dy = iy + .5 - 40.75
    Z = 5.008122486108
    D, _ = oracle.density_exact([[302, 306, 342, 346]], 640, 640, 8, 2.0)
    for iy, ix in [(40, 40), (38, 43), (34, 46), (46, 34), (47, 40), (40, 33)]:
        dx, dy = ix + 0.5 - 40.25, iy + 0.5 - 40.75
        want = math.exp(-(dx * dx + dy * dy) / 8.0) / (Z * Z) if (abs(dx) <= 6 and abs(dy) <= 6) else 0.0
        assert D[iy, ix] == pytest.approx(want, rel=2e-6, abs=1e-12)
    assert D[40, 33] == 0.0 and D[47, 40] == 0.0            # |dx| = 6.75 > 6, |dy| = 6.75 > 6
    # the binned grid puts this bird in cell (40, 40): the two differ, by design (A14 vs B4)
    Db, _ = oracle.density([[302, 306, 342, 346]], 640, 640, 8, 2.0)
    assert abs(D - Db).max() > 1e-3


def test_density_exact_brute_force_and_no_fold_at_the_border():
    rng = np.random.default_rng(2)
    W, H, cell, sigma = 160, 96, 8, 2.5
    c = np.stack([rng.uniform(-10, W + 10, 40), rng.uniform(-10, H + 10, 40)], 1)
    boxes = np.concatenate([c - 7.3, c + 7.3], 1).astype(np.float32)
    D, n_in = oracle.density_exact(boxes, W, H, cell, sigma)
    R, w = oracle.taps(sigma)
    Z = float(np.exp(-np.arange(-R, R + 1) ** 2 / (2 * sigma * sigma)).sum())
    cx = (boxes[:, 0] + boxes[:, 2]) * np.float32(0.5); cy = (boxes[:, 1] + boxes[:, 3]) * np.float32(0.5)
    ok = (cx >= 0) & (cx < W) & (cy >= 0) & (cy < H)
    assert n_in == int(ok.sum())
    iy, ix = np.mgrid[0:H // cell, 0:W // cell]
    ref = np.zeros((H // cell, W // cell))
    for x, y in zip(cx[ok], cy[ok]):                         # numpy restatement: vectorised over cells ("cdist")
        dx = (ix + 0.5).astype(np.float32) - np.float32(x / np.float32(cell)); dy = (iy + 0.5).astype(np.float32) - np.float32(y / np.float32(cell))
        m = (np.abs(dx) <= R) & (np.abs(dy) <= R)
        ref += np.where(m, np.exp(-(dx.astype(np.float64) ** 2 + dy.astype(np.float64) ** 2) / (2 * sigma * sigma)) / Z ** 2, 0.0)
    np.testing.assert_allclose(D, ref, rtol=1e-6, atol=1e-12)
    # mass is NOT conserved near the border (no fold): a bird in the corner cell keeps about a quarter of its mass
    Dc, _ = oracle.density_exact([[0, 0, 8, 8]], W, H, cell, sigma)
    assert 0.2 < float(Dc.sum()) < 0.35


# ---------------------------------------------------------------- f4: pre-processing (B6)
@pytest.mark.parametrize("src,dst", [((54, 96), (32, 64)), ((36, 64), (72, 128)), ((45, 80), (45, 80)), ((108, 192), (40, 40))])
def test_preprocess_against_torch_interpolate(src, dst):
    import torch
    import flockgen
    img = flockgen.make_image_batch(1, src[1], src[0], seed=9)[0]
    mean, std = [0.485, 0.456, 0.406], [0.229, 0.224, 0.225]
    got = oracle.preprocess(img, dst[0], dst[1], mean, std)
    t = torch.from_numpy(img.astype(np.float64)).permute(2, 0, 1)[None]
    ref = torch.nn.functional.interpolate(t, size=dst, mode="bilinear", align_corners=False, antialias=False)[0].numpy()
    ref = (ref / 255.0 - np.array(mean, dtype=np.float32).astype(np.float64)[:, None, None]) / np.array(std, dtype=np.float32).astype(np.float64)[:, None, None]
    np.testing.assert_allclose(got, ref, rtol=1e-9, atol=1e-9)


def test_preprocess_identity_and_constant_image():
    img = np.arange(5 * 7 * 3, dtype=np.uint8).reshape(5, 7, 3)
    got = oracle.preprocess(img, 5, 7, [0, 0, 0], [1, 1, 1])
    np.testing.assert_allclose(got, img.transpose(2, 0, 1) / 255.0, rtol=0, atol=1e-15)      # same size: exact copy, CHW
    const = np.full((9, 11, 3), 200, dtype=np.uint8)
    got = oracle.preprocess(const, 4, 23, [0.5, 0.25, 0.0], [0.5, 2.0, 1.0])
    np.testing.assert_allclose(got[0], (200 / 255 - 0.5) / 0.5, rtol=1e-12)
    np.testing.assert_allclose(got[1], (200 / 255 - 0.25) / 2.0, rtol=1e-12)
    # 2x upscale of a two-pixel ramp by hand: src centres at 0.5, 1.5 -> dst centres 0.25, 0.75, 1.25, 1.75 -> 0, .25, .75, 1
    ramp = np.zeros((1, 2, 3), dtype=np.uint8); ramp[0, 1] = 255
    got = oracle.preprocess(ramp, 1, 4, [0, 0, 0], [1, 1, 1])
    np.testing.assert_allclose(got[0, 0], [0.0, 0.25, 0.75, 1.0], atol=1e-15)
