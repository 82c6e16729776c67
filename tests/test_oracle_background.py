"""Pins of the background-map / source-detection oracle (oracle/background.py).

The paper prints no formula or worked value for these two stages (PAPER.md:193-194 name them only), so the oracle is
pinned against what the mathematics fixes: the standard library's median on tiny cells, closed forms for constant and
planar images, Gaussian statistics, the outlier-rejection property of a 3x3 median, and hand-built sources whose
detection, tie-breaking, flux and centroid follow from the definitions by inspection.
"""
import statistics

import numpy as np
import pytest

from oracle import background as ob


def test_median_rule_against_stdlib_and_hand_values():
    rng = np.random.default_rng(1)
    for n in (1, 2, 3, 4, 7, 16, 33, 64):
        v = rng.normal(size=n)
        assert ob.median_rule(v) == pytest.approx(statistics.median(v.tolist()), abs=0, rel=1e-15)
    assert ob.median_rule([3.0, 1.0, 2.0]) == 2.0
    assert ob.median_rule([4.0, 1.0, 3.0, 2.0]) == 2.5        # mean of the two central values, not the lower one
    assert ob.median_rule([5.0, 5.0, 1.0, 9.0]) == 5.0


def test_cell_stats_brute_force_with_masks_and_ragged_cells():
    rng = np.random.default_rng(2)
    H, W, B = 21, 27, 8                                   # ragged right column (3 px) and bottom row (5 px)
    cal = rng.normal(100.0, 5.0, (H, W))
    mask = (rng.random((H, W)) > 0.2).astype(np.uint8)
    mask[0:8, 0:8] = 0                                    # a fully masked cell
    med, sig, valid, n_good = ob.cell_stats(cal, mask, B=B, n_min=4)
    assert med.shape == (3, 4)
    assert not valid[0, 0] and med[0, 0] == 0 and sig[0, 0] == 0 and n_good[0, 0] == 0
    for gy in range(3):
        for gx in range(4):
            vals = [cal[y, x] for y in range(gy * B, min(gy * B + B, H)) for x in range(gx * B, min(gx * B + B, W))
                    if mask[y, x]]
            assert n_good[gy, gx] == len(vals)
            assert valid[gy, gx] == (len(vals) >= 4)
            if valid[gy, gx]:
                m = statistics.median(vals)
                assert med[gy, gx] == pytest.approx(m, rel=1e-15)
                assert sig[gy, gx] == pytest.approx(1.4826 * statistics.median([abs(v - m) for v in vals]), rel=1e-14)


def test_constant_image_gives_constant_background_zero_noise_no_sources():
    cal = np.full((96, 130), 37.5)
    mask = np.ones(cal.shape, np.uint8)
    bkg, nse = ob.background(cal, mask, B=32)
    assert np.all(bkg == 37.5) and np.all(nse == 0.0)
    bmap, und = ob.interp_grid(bkg, 130, 96, B=32)
    assert np.all(bmap == 37.5) and not und.any()
    assert ob.detect(cal, mask, bkg, nse, B=32)["x"].size == 0      # s = 0 is not > 0


def test_plane_is_reproduced_away_from_the_grid_border():
    # a + b x + c y over full cells: each cell's values are symmetric about the value at the cell centre, the 3x3
    # median of a planar grid is its centre value, and bilinear interpolation between centres is exact for a plane.
    B, GX, GY = 16, 6, 5
    W, H = GX * B, GY * B
    y, x = np.mgrid[0:H, 0:W]
    plane = 50.0 + 0.25 * x - 0.125 * y
    med, sig, valid, _ = ob.cell_stats(plane, np.ones((H, W), np.uint8), B=B)
    cx = np.arange(GX) * B + (B - 1) / 2.0
    cy = np.arange(GY) * B + (B - 1) / 2.0
    assert np.allclose(med, 50.0 + 0.25 * cx[None, :] - 0.125 * cy[:, None], atol=1e-12)
    bkg, nse = ob.filter_grid(med, sig, valid)
    assert np.allclose(bkg[1:-1, 1:-1], med[1:-1, 1:-1], atol=1e-12)
    bmap, _ = ob.interp_grid(bkg, W, H, B=B)
    x0, x1 = int(cx[1]) + 1, int(cx[-2])
    y0, y1 = int(cy[1]) + 1, int(cy[-2])
    assert np.allclose(bmap[y0:y1, x0:x1], plane[y0:y1, x0:x1], atol=1e-11)
    # x and y are not interchangeable: the slopes differ in sign
    assert bmap[y0, x1 - 1] > bmap[y0, x0] and bmap[y1 - 1, x0] < bmap[y0, x0]


def test_interp_nodes_and_clamping():
    grid = np.array([[1.0, 2.0, 4.0], [8.0, 16.0, 32.0]])
    B = 4
    m, und = ob.interp_grid(grid, 12, 8, B=B)
    assert not und.any()
    # centres at 1.5, 5.5, 9.5: pixel 1 and 2 straddle the first centre; left of it the map is clamped
    assert m[0, 0] == m[0, 1] == 1.0 and m[7, 11] == 32.0
    assert m[0, 2] == pytest.approx(1.0 + (2.0 - 1.5) / 4 * (2.0 - 1.0))      # row 0 is above the first row centre
    assert m[3, 0] == pytest.approx(1.0 + (3.0 - 1.5) / 4 * (8.0 - 1.0))
    assert m[3, 7] == pytest.approx((1 - .375) * ((1 - .375) * 2 + .375 * 4) + .375 * ((1 - .375) * 16 + .375 * 32))
    # a non-finite node makes every pixel that uses it undefined, zero weight included (clamped pixels x <= 1 use
    # nodes 0 and 1 with t = 0): centres 1.5, 5.5, 9.5, 13.5, node 1 is used by x <= 9
    grid = np.array([[1.0, np.inf, 4.0, 5.0], [8.0, 16.0, 32.0, 64.0]])
    m, und = ob.interp_grid(grid, 16, 8, B=B)
    assert und[:, :10].all() and not und[:, 10:].any()
    assert np.isinf(m[und]).all() and np.isfinite(m[~und]).all()


def test_gaussian_noise_statistics():
    rng = np.random.default_rng(3)
    cal = rng.normal(200.0, 14.0, (256, 256))
    med, sig, valid, _ = ob.cell_stats(cal, np.ones(cal.shape, np.uint8), B=64)
    assert valid.all()
    # median of 4096 normals: sd = 1.2533 * 14 / 64 = 0.274; 1.4826 * MAD -> sigma with sd ~ 1.17 %
    assert np.all(np.abs(med - 200.0) < 5 * 0.274)
    assert np.all(np.abs(sig / 14.0 - 1.0) < 0.06)


def test_three_by_three_median_removes_a_single_outlier_cell():
    rng = np.random.default_rng(4)
    med = rng.normal(100.0, 0.1, (6, 7)); sig = rng.normal(5.0, 0.01, (6, 7))
    valid = np.ones((6, 7), bool)
    b0, n0 = ob.filter_grid(med, sig, valid)
    med2 = med.copy(); med2[3, 3] += 1000.0
    b1, _ = ob.filter_grid(med2, sig, valid)
    assert np.abs(b1 - b0).max() < 0.3          # the outlier never becomes a median; ranks shift by at most one
    assert abs(b1[3, 3] - 100.0) < 0.5
    # an invalid cell is ignored and filled from its neighbours; an isolated grid is undefined
    valid2 = valid.copy(); valid2[0, 0] = False
    b2, n2 = ob.filter_grid(med, sig, valid2)
    assert np.isfinite(n2).all() and b2[0, 0] == pytest.approx(ob.median_rule([med[0, 1], med[1, 0], med[1, 1]]))
    b3, n3 = ob.filter_grid(med[:1, :1], sig[:1, :1], np.zeros((1, 1), bool))
    assert b3[0, 0] == 0.0 and np.isinf(n3[0, 0])


def _detect_on_zero_background(cal, mask=None, B=16, k=5.0):
    mask = np.ones(cal.shape, np.uint8) if mask is None else mask
    bkg, nse = ob.background(cal, mask, B=B)
    return ob.detect(cal, mask, bkg, nse, B=B, k_sigma=k), bkg, nse


def test_hand_built_sources_position_flux_centroid_and_ties():
    cal = np.zeros((48, 64))
    cal[10, 20] = 100.0                         # single pixel
    cal[30, 40] = cal[30, 41] = 50.0            # horizontal tie: the raster-first pixel (x = 40) wins, cx = +1/2
    cal[20, 8] = cal[21, 8] = 30.0              # vertical tie: the upper pixel (y = 20) wins, cy = +1/2
    cal[40, 50] = 80.0; cal[40, 51] = 20.0      # asymmetric pair: cx = 20 / 100
    d, bkg, nse = _detect_on_zero_background(cal)
    assert np.all(bkg == 0) and np.all(nse == 0)
    assert list(zip(d["y"], d["x"])) == [(10, 20), (20, 8), (30, 40), (40, 50)]      # catalogue order
    assert np.allclose(d["peak"], [100, 30, 50, 80]) and np.allclose(d["flux"], [100, 60, 100, 100])
    assert np.allclose(d["cx"], [0, 0, 0.5, 0.2]) and np.allclose(d["cy"], [0, 0.5, 0, 0])
    assert d["strict"].all()


def test_masked_pixels_neither_win_nor_count_and_borders_work():
    cal = np.zeros((32, 32)); mask = np.ones((32, 32), np.uint8)
    cal[5, 5] = 100.0; mask[5, 5] = 0           # a masked peak is not a source ...
    cal[5, 6] = 40.0                            # ... and does not suppress or feed its good neighbour
    cal[0, 0] = 10.0; cal[31, 31] = 7.0         # frame corners: off-frame neighbours are ignored
    d, _, _ = _detect_on_zero_background(cal, mask)
    assert list(zip(d["y"], d["x"])) == [(0, 0), (5, 6), (31, 31)]
    assert np.allclose(d["flux"], [10, 40, 7]) and np.allclose(d["cx"], 0) and np.allclose(d["cy"], 0)


def test_threshold_uses_interpolated_noise_and_margins_are_reported():
    rng = np.random.default_rng(5)
    H, W, B = 128, 128, 32
    cal = rng.normal(100.0, 4.0, (H, W))
    cal[64, 64] = 100.0 + 4.0 * 12              # 12 sigma: found
    cal[19:22, 89:92] = 100.0
    cal[20, 90] = 100.0 + 4.0 * 3               # 3 sigma above quiet neighbours: not found at k = 5
    mask = np.ones((H, W), np.uint8)
    bkg, nse = ob.background(cal, mask, B=B)
    d = ob.detect(cal, mask, bkg, nse, B=B, k_sigma=5.0)
    found = set(zip(d["y"].tolist(), d["x"].tolist()))
    assert (64, 64) in found and (20, 90) not in found
    assert len(found) <= 2                      # 5-sigma noise peaks: 16384 * 2.9e-7 expected
    i = list(zip(d["y"].tolist(), d["x"].tolist())).index((64, 64))
    assert d["m_thr"][i] == pytest.approx(d["peak"][i] - 5.0 * d["nse"][i]) and d["m_max"][i] > 20
    assert abs(d["bkg"][i] - 100.0) < 1.0 and abs(d["nse"][i] - 4.0) < 0.5
    # lowering k to 2.5 finds the 3-sigma pixel too; slack returns a superset with the strict flag
    d2 = ob.detect(cal, mask, bkg, nse, B=B, k_sigma=2.5)
    assert (20, 90) in set(zip(d2["y"].tolist(), d2["x"].tolist()))
    d3 = ob.detect(cal, mask, bkg, nse, B=B, k_sigma=5.0, slack=1.0)
    assert d3["x"].size >= d["x"].size and int(d3["strict"].sum()) == d["x"].size


def test_undefined_background_suppresses_detection():
    cal = np.zeros((32, 64)); mask = np.ones((32, 64), np.uint8)
    mask[:, 32:] = 0; mask[4, 40] = 1; cal[4, 40] = 500.0      # right half: one good pixel < n_min per cell
    cal[8, 8] = 9.0
    bkg, nse = ob.background(cal, mask, B=16, n_min=16)
    assert np.isinf(nse[:, 3]).all() and np.isfinite(nse[:, :3]).all()     # column 2 borrows from column 1
    d = ob.detect(cal, mask, bkg, nse, B=16)
    assert list(zip(d["y"], d["x"])) == [(8, 8)]


def test_gaussian_star_found_at_its_peak_pixel_with_signed_centroid():
    y, x = np.mgrid[0:64, 0:64]
    sig = 2.0 / 2.3548
    star = lambda x0, y0, f: f * np.exp(-((x - x0) ** 2 + (y - y0) ** 2) / (2 * sig * sig))
    cal = star(20.3, 30.0, 1000.0) + star(45.0, 12.8, 400.0)
    d, _, _ = _detect_on_zero_background(cal, k=5.0)
    assert list(zip(d["y"], d["x"])) == [(13, 45), (30, 20)]
    assert d["cx"][1] > 0.05 and abs(d["cy"][1]) < 1e-12 and d["cy"][0] < -0.05 and abs(d["cx"][0]) < 1e-12


def test_catalogue_order_is_raster():
    """R-D6: ascending y * W + x, whatever tiling an implementation uses (the points straddle 64 x 32 blocks)."""
    cal = np.zeros((70, 200))
    for (y, x) in [(2, 150), (3, 10), (31, 70), (33, 5), (40, 199), (69, 64)]:
        cal[y, x] = 10.0 + x
    mask = np.ones(cal.shape, np.uint8)
    bkg, nse = ob.background(cal, mask, B=16)
    d = ob.detect(cal, mask, bkg, nse, B=16)
    assert list(zip(d["y"], d["x"])) == [(2, 150), (3, 10), (31, 70), (33, 5), (40, 199), (69, 64)]
    key = d["y"].astype(np.int64) * 200 + d["x"]
    assert np.all(np.diff(key) > 0)
