"""Pins of oracle/subtract.py (direct image subtraction per tile).  The paper
prints no formula (the method is in its ref [17]); each reading R-X1 .. R-X8 is pinned by something other than the
oracle's own code: library least squares, hand-computed values, symmetries (identical images, linearity), brute force
over Python loops, and the C oracle's nested <-> (ix, iy) mapping."""
import numpy as np
import pytest

import oracle
from oracle import subtract as osub

SIDE = 32
PPT = SIDE * SIDE


def _pair(img_s, img_r, w_s=None, w_r=None):
    """Grid images [iy][ix] -> one-tile (sum, wsum) pairs in nested order."""
    w_s = np.ones_like(img_s) if w_s is None else w_s
    w_r = np.full_like(img_r, 30.0) if w_r is None else w_r
    return (osub.grid_to_tile(img_s * w_s), osub.grid_to_tile(w_s), osub.grid_to_tile(img_r * w_r), osub.grid_to_tile(w_r))


def _smooth(seed=0, side=SIDE):
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:side, 0:side]
    img = 200.0 + 0.7 * x - 0.4 * y
    for _ in range(5):
        cx, cy, a = rng.uniform(3, side - 3), rng.uniform(3, side - 3), rng.uniform(200, 3000)
        img = img + a * np.exp(-((x - cx) ** 2 + (y - cy) ** 2) / (2 * 0.85 ** 2))
    return img


def test_nested_grid_mapping_matches_the_c_oracle():
    """ix = even bits, iy = odd bits: against orc_nest2xyf (pinned in test_oracle_healpix.py) for every in-tile index."""
    ix, iy = osub.deinterleave(np.arange(4096), 6)
    for q in list(range(0, 4096, 37)) + [4095]:
        f, x, y = oracle.nest2xyf(64, 5 * 4096 + q)
        assert (f, x, y) == (5, ix[q], iy[q])
    g = np.arange(PPT).reshape(SIDE, SIDE)
    assert np.array_equal(osub.tile_to_grid(osub.grid_to_tile(g), SIDE), g)


@pytest.mark.parametrize("match", [osub.MATCH_NONE, osub.MATCH_AFFINE])
def test_identical_images_give_zero_difference_and_no_candidate(match):
    img = _smooth(1)
    ss, sw, rs, rw = _pair(img, img)
    out = osub.subtract_tiles([7], PPT, 1 << 10, ss, sw, rs, rw, match=match)
    assert abs(out["alpha"][0] - 1) < 1e-12 and abs(out["beta"][0]) < 1e-9
    assert np.all(np.abs(out["diff"]) < 1e-9) and np.all(np.abs(out["sig"]) < 1e-9)
    assert out["cat"]["pixel"].size == 0 and out["n_valid"][0] == PPT


def test_affine_match_is_library_least_squares():
    rng = np.random.default_rng(2)
    r = _smooth(3)
    s = 0.83 * r + 12.5 + rng.normal(0, 3.0, r.shape)
    ws = (rng.random(r.shape) > 0.1).astype(float)            # 10 % of the science pixels are invalid
    ss, sw, rs, rw = _pair(s, r, w_s=ws)
    out = osub.subtract_tiles([0], PPT, 1 << 10, ss, sw, rs, rw)
    v = ws > 0
    a, b = np.polyfit(r[v], s[v], 1)
    assert abs(out["alpha"][0] - a) < 1e-10 and abs(out["beta"][0] - b) < 1e-8 and out["n_valid"][0] == v.sum()
    # residuals of a least-squares line sum to zero and are orthogonal to the regressor
    d = osub.tile_to_grid(out["diff"], SIDE)
    assert abs(d[v].sum()) < 1e-7 and abs((d[v] * r[v]).sum()) < 1e-4
    assert np.all(d[~v] == 0)


def test_match_fallbacks():
    r = np.full((SIDE, SIDE), 100.0)                            # constant reference: the slope is undetermined
    s = r + 5.0
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s, r))
    assert out["alpha"][0] == 1.0 and abs(out["beta"][0] - 5.0) < 1e-12 and np.all(np.abs(out["diff"]) < 1e-12)
    # constant up to float32 rounding (sum / wsum of a float32 coadd): still no slope to fit
    wr = np.random.default_rng(0).uniform(20, 30, r.shape).astype(np.float32)
    rs32 = (np.float32(100.0) * wr).astype(np.float32)
    rq = (rs32 / wr).astype(np.float64)
    assert rq.std() > 0
    out = osub.subtract_tiles([0], PPT, 1 << 10, osub.grid_to_tile(s), osub.grid_to_tile(np.ones_like(s)), osub.grid_to_tile(rs32), osub.grid_to_tile(wr))
    assert out["alpha"][0] == 1.0 and abs(out["beta"][0] - 5.0) < 1e-4
    ws = np.zeros((SIDE, SIDE)); ws[0, :10] = 1.0               # 10 valid pixels < n_min = 16
    r2 = _smooth(4)
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(2 * r2, r2, w_s=ws))
    assert out["alpha"][0] == 1.0 and abs(out["beta"][0] - r2[0, :10].mean()) < 1e-9 and out["n_valid"][0] == 10
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(r2, r2, w_s=np.zeros((SIDE, SIDE))))
    assert (out["alpha"][0], out["beta"][0], out["n_valid"][0]) == (1.0, 0.0, 0) and out["cat"]["pixel"].size == 0


def test_noise_and_significance_by_hand():
    """R-X4 / R-X5 at one pixel, numbers worked by hand: m = 400, read noise 2, gain 0.5 => one exposure's variance
    4 + 800 = 804; science weight 1, reference weight 4, alpha = 1 => sigma^2 = 804 * 1.25 = 1005; d = 63.4."""
    r = np.full((SIDE, SIDE), 400.0)
    s = r.copy(); s[10, 20] += 63.4
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s, r, w_r=np.full_like(r, 4.0)), match=osub.MATCH_NONE,
                              read_noise=2.0, gain=0.5, k_sigma=1.5)
    c = out["cat"]
    assert c["pixel"].size == 1
    assert abs(c["noise"][0] - np.sqrt(1005.0)) < 1e-12 and abs(c["sig"][0] - 63.4 / np.sqrt(1005.0)) < 1e-12
    assert abs(c["diff"][0] - 63.4) < 1e-12 and abs(c["flux"][0] - 63.4) < 1e-12
    ix, iy = osub.deinterleave(c["pixel"] % PPT, 5)
    assert (ix[0], iy[0]) == (20, 10)
    # a negative prediction contributes no Poisson term: sigma^2 = rn^2 (1 + 1/4)
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s - 500.0, r - 500.0, w_r=np.full_like(r, 4.0)), match=osub.MATCH_NONE,
                              read_noise=2.0, gain=0.5, k_sigma=1.5)
    assert abs(out["cat"]["noise"][0] - np.sqrt(4.0 * 1.25)) < 1e-12


def test_injected_transient_is_the_one_candidate_with_its_flux():
    """PAPER.md:169 (Fig. 3): a science segment = scaled reference + sky offset + an injected point source.  The affine
    match recovers scale and offset, the difference holds the source alone, and the 3 x 3 flux is the injected one."""
    r = _smooth(5)
    y, x = np.mgrid[0:SIDE, 0:SIDE]
    psf = np.exp(-((x - 13) ** 2 + (y - 21) ** 2) / (2 * 0.6 ** 2))
    psf /= psf.sum()
    F = 900.0
    s = 0.9 * r + 7.0 + F * psf
    out = osub.subtract_tiles([3], PPT, 1 << 10, *_pair(s, r), k_sigma=5.0)
    assert abs(out["alpha"][0] - 0.9) < 2e-3 and abs(out["beta"][0] - 7.0) < 2.0     # the source biases the fit slightly
    c = out["cat"]
    assert c["pixel"].size == 1 and c["tile_rank"][0] == 0
    ix, iy = osub.deinterleave(c["pixel"] % PPT, 5)
    assert (ix[0], iy[0]) == (13, 21) and c["pixel"][0] // PPT == 3
    win = (np.abs(x - 13) <= 1) & (np.abs(y - 21) <= 1)
    assert abs(c["flux"][0] - F * psf[win].sum()) < 0.02 * F and c["sig"][0] > 5
    # without the source: nothing
    out0 = osub.subtract_tiles([3], PPT, 1 << 10, *_pair(0.9 * r + 7.0, r))
    assert out0["cat"]["pixel"].size == 0 and np.abs(out0["diff"]).max() < 1e-9


def test_difference_is_linear_in_the_science_image():
    """Affine match: s -> c s + e maps (alpha, beta, d) -> (c alpha, c beta + e, c d)."""
    rng = np.random.default_rng(6)
    r = _smooth(7)
    s = 1.1 * r - 3.0 + rng.normal(0, 4.0, r.shape)
    a = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s, r))
    b = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(2.5 * s + 40.0, r))
    assert abs(b["alpha"][0] - 2.5 * a["alpha"][0]) < 1e-10 and abs(b["beta"][0] - (2.5 * a["beta"][0] + 40.0)) < 1e-8
    assert np.allclose(b["diff"], 2.5 * a["diff"], rtol=0, atol=1e-8)


def test_masked_pixels_are_never_candidates_and_do_not_count_as_neighbours():
    r = np.full((SIDE, SIDE), 300.0)
    s = r.copy()
    s[5, 5] += 500.0; s[5, 6] += 800.0            # the brighter neighbour is masked: (5, 5) must still be found
    s[20, 20] += 900.0                            # masked peak: never a candidate
    s[12, 12] += 400.0                            # reference invalid there
    ws = np.ones((SIDE, SIDE)); ws[5, 6] = 0.0; ws[20, 20] = 0.2      # 0.2 < sci_wmin = 0.5
    wr = np.full((SIDE, SIDE), 30.0); wr[12, 12] = 0.0
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s, r, ws, wr), match=osub.MATCH_NONE)
    ix, iy = osub.deinterleave(out["cat"]["pixel"] % PPT, 5)
    assert list(zip(iy.tolist(), ix.tolist())) == [(5, 5)]
    d = osub.tile_to_grid(out["diff"], SIDE)
    assert d[5, 6] == 0 and d[20, 20] == 0 and d[12, 12] == 0 and out["n_valid"][0] == PPT - 3
    assert abs(out["cat"]["flux"][0] - 500.0) < 1e-9       # the masked neighbour's 800 is not in the 3 x 3 flux


def test_tie_rule_tile_edges_and_order():
    """Equal neighbours: the smaller nested index is the candidate.  Neighbours beyond the tile do not exist (tiles are
    independent).  Catalogue order = ascending nested pixel index across tiles."""
    r = np.full((SIDE, SIDE), 300.0)
    s = r.copy()
    s[8, 8] += 500.0; s[8, 9] += 500.0            # nested(8, 8) < nested(9, 8) [ix = 9 sets a lower bit]: (8, 8) wins
    s[0, 0] += 450.0                              # tile corner
    s[31, 31] += 470.0                            # opposite corner
    ss, sw, rs, rw = _pair(s, r)
    z = np.zeros(PPT); rwz = np.full(PPT, 30.0)
    s2 = r.copy(); s2[3, 4] += 600.0
    ss2, sw2, rs2, rw2 = _pair(s2, r)
    cat = lambda *a: np.concatenate(a)
    out = osub.subtract_tiles([11, 40], PPT, 1 << 10, cat(ss2, ss), cat(sw2, sw), cat(rs2, rs), cat(rw2, rw), match=osub.MATCH_NONE)
    c = out["cat"]
    assert np.all(np.diff(c["pixel"]) > 0)
    ix, iy = osub.deinterleave(c["pixel"] % PPT, 5)
    got = list(zip((c["pixel"] // PPT).tolist(), iy.tolist(), ix.tolist()))
    assert got == [(11, 3, 4), (40, 0, 0), (40, 8, 8), (40, 31, 31)]
    assert c["tile_rank"].tolist() == [0, 1, 1, 1]
    # vertical tie: nested(8, 8) vs nested(8, 9) in (ix, iy) -- the iy bit is the higher one, so (iy 8) wins again
    s3 = r.copy(); s3[8, 8] += 500.0; s3[9, 8] += 500.0
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s3, r), match=osub.MATCH_NONE)
    ix, iy = osub.deinterleave(out["cat"]["pixel"] % PPT, 5)
    assert list(zip(iy.tolist(), ix.tolist())) == [(8, 8)]


def test_detection_against_a_python_loop():
    """R-X6 by brute force over Python loops on a noisy tile (different code: dictionaries and scalar comparisons)."""
    rng = np.random.default_rng(8)
    r = _smooth(9)
    s = r + rng.normal(0, 15.0, r.shape)
    ws = (rng.random(r.shape) > 0.05).astype(float)
    out = osub.subtract_tiles([0], PPT, 1 << 10, *_pair(s, r, w_s=ws), match=osub.MATCH_NONE, k_sigma=2.0)
    S = osub.tile_to_grid(out["sig"], SIDE)
    q = osub.tile_to_grid(np.arange(PPT), SIDE)
    want = []
    for y in range(SIDE):
        for x in range(SIDE):
            if ws[y, x] == 0 or not S[y, x] > 2.0:
                continue
            ok = True
            for dy in (-1, 0, 1):
                for dx in (-1, 0, 1):
                    yy, xx = y + dy, x + dx
                    if (dy or dx) and 0 <= yy < SIDE and 0 <= xx < SIDE and ws[yy, xx] > 0:
                        if q[yy, xx] < q[y, x]:
                            ok = ok and S[y, x] > S[yy, xx]
                        else:
                            ok = ok and S[y, x] >= S[yy, xx]
            if ok:
                want.append(int(q[y, x]))
    assert sorted(want) == out["cat"]["pixel"].tolist() and len(want) > 5
