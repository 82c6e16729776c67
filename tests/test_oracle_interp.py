"""Pins P7 for O1 (calibration) and O6 (interpolation): closed forms and special cases that reduce to
textbook results (BASELINE.json north_star: "exact reproduction of constant and linear-gradient images
under bilinear interpolation")."""
import math

import numpy as np
import pytest

import oracle


def _img(H=24, W=32, seed=0):
    rng = np.random.default_rng(seed)
    return rng.uniform(100, 60000, (H, W)), np.ones((H, W), np.uint8)


def test_o1_calibration_closed_form_and_mask():
    raw = np.array([[1200, 65535, 1500, 900], [1000, 2000, 3000, 65534]], dtype=np.uint16)
    bias = np.full((2, 4), 1000.0, np.float32)
    dark = np.full((2, 4), 0.5, np.float32)
    flat = np.array([[1.0, 1.0, 0.5, 2.0], [0.05, np.nan, 1.25, 1.0]], np.float32)
    bpm = np.zeros((2, 4), np.uint8)
    bpm[0, 3] = 7
    cal, m = oracle.calibrate(raw, bias, dark, flat, bpm, t_exp=10.0, sat_adu=65535, flat_min=0.1)
    # (raw - 1000 - 0.5*10)/flat
    assert m.tolist() == [[1, 0, 1, 0], [0, 0, 1, 1]]
    assert cal[0, 0] == 195.0 and cal[0, 2] == 990.0 and cal[1, 2] == 1596.0 and cal[1, 3] == 64529.0
    assert cal[0, 1] == 0 and cal[0, 3] == 0 and cal[1, 0] == 0 and cal[1, 1] == 0
    # negative calibrated values are kept (no clamp)
    cal2, m2 = oracle.calibrate(np.array([[900]], np.uint16), bias[:1, :1], dark[:1, :1], flat[:1, :1], None, 10.0)
    assert cal2[0, 0] == -105.0 and m2[0, 0] == 1
    # non-finite masters mask the pixel
    b2 = bias[:1, :1].copy()
    b2[0, 0] = np.inf
    assert oracle.calibrate(np.array([[900]], np.uint16), b2, dark[:1, :1], flat[:1, :1], None, 10.0)[1][0, 0] == 0


@pytest.mark.parametrize("kernel", [oracle.BILINEAR, oracle.LANCZOS3])
def test_p7_integer_positions_return_the_pixel(kernel):
    cal, m = _img()
    for (i, j) in [(5, 5), (10, 7), (20, 15), (3, 3)]:
        v, w, _ = oracle.interp(cal, m, float(i), float(j), kernel)
        assert abs(v - cal[j, i]) < 1e-9 * cal[j, i] and w == 1.0


@pytest.mark.parametrize("kernel", [oracle.BILINEAR, oracle.LANCZOS3])
def test_p7_constant_image_also_beside_masks(kernel):
    cal = np.full((24, 32), 777.25)
    m = np.ones((24, 32), np.uint8)
    m[10, 12] = 0
    m[:, 20] = 0
    rng = np.random.default_rng(1)
    nz = 0
    for _ in range(500):
        x, y = rng.uniform(3, 28), rng.uniform(3, 20)
        v, w, _ = oracle.interp(cal, m, x, y, kernel, w_min=0.3)
        if w > 0:
            nz += 1
            assert abs(v - 777.25) < 1e-9
            assert 0.3 <= w <= 1.0
        else:
            assert v == 0.0
    assert nz > 300


def test_p7_bilinear_reproduces_linear_gradient_exactly():
    H, W = 24, 32
    yy, xx = np.mgrid[0:H, 0:W]
    cal = 3.0 + 0.5 * xx - 1.25 * yy
    m = np.ones((H, W), np.uint8)
    rng = np.random.default_rng(2)
    for _ in range(500):
        x, y = rng.uniform(0, W - 1), rng.uniform(0, H - 1)
        v, w, _ = oracle.interp(cal, m, x, y, oracle.BILINEAR)
        assert w == 1.0
        assert abs(v - (3.0 + 0.5 * x - 1.25 * y)) < 1e-11


def test_p7_bilinear_closed_form_and_axis_order():
    """cal[j][i] with i <-> x (fast axis): a transposed operand fails here."""
    cal = np.zeros((8, 8))
    cal[2, 5] = 100.0  # y = 2, x = 5
    m = np.ones((8, 8), np.uint8)
    v, w, _ = oracle.interp(cal, m, 4.75, 2.0, oracle.BILINEAR)
    assert abs(v - 75.0) < 1e-12
    v, w, _ = oracle.interp(cal, m, 5.0, 1.5, oracle.BILINEAR)
    assert abs(v - 50.0) < 1e-12
    v, w, _ = oracle.interp(cal, m, 5.25, 2.5, oracle.BILINEAR)
    assert abs(v - 100 * 0.75 * 0.5) < 1e-12
    v, w, _ = oracle.interp(cal, m, 2.0, 5.0, oracle.BILINEAR)
    assert v == 0.0


def test_p7_lanczos3_kernel_values():
    """Delta image => the interpolant IS the (normalised) separable kernel: check against
    L(t) = sinc(t) sinc(t/3) evaluated with math.sin here, incl. the negative lobe and |t| >= 3 cut."""
    cal = np.zeros((16, 16))
    cal[8, 8] = 1.0
    m = np.ones((16, 16), np.uint8)

    def L(t):
        if t == 0:
            return 1.0
        if abs(t) >= 3:
            return 0.0
        return math.sin(math.pi * t) / (math.pi * t) * math.sin(math.pi * t / 3) / (math.pi * t / 3)

    for dx, dy in [(0.5, 0.0), (1.5, 0.0), (0.25, 0.75), (-2.6, 0.3), (2.9, -2.9), (-1.2, 1.7)]:
        x, y = 8 + dx, 8 + dy
        v, w, _ = oracle.interp(cal, m, x, y, oracle.LANCZOS3)
        i0, j0 = math.floor(x), math.floor(y)
        sx = sum(L(x - i) for i in range(i0 - 2, i0 + 4))
        sy = sum(L(y - j) for j in range(j0 - 2, j0 + 4))
        assert abs(v - L(dx) * L(dy) / (sx * sy)) < 1e-14
        assert w == 1.0
    assert L(1.5) < 0  # negative lobe kept (no clamping)
    # outside the 6x6 support the delta does not contribute
    assert oracle.interp(cal, m, 8 + 3.2, 8.0, oracle.LANCZOS3)[0] == 0.0


def test_p7_weight_is_good_kernel_mass_and_wmin_rule():
    cal, m = _img()
    m[6, 6] = 0
    # bilinear at (5.25, 5.5): taps (5,5),(6,5),(5,6),(6,6) with weights .75*.5,.25*.5,.75*.5,.25*.5
    v, w, _ = oracle.interp(cal, m, 5.25, 5.5, oracle.BILINEAR, w_min=0.5)
    assert abs(w - (1 - 0.125)) < 1e-15
    exp = (0.375 * cal[5, 5] + 0.125 * cal[5, 6] + 0.375 * cal[6, 5]) / 0.875
    assert abs(v - exp) < 1e-9
    # strict rule: w_min = 1 rejects any bad tap
    assert oracle.interp(cal, m, 5.25, 5.5, oracle.BILINEAR, w_min=1.0)[:2] == (0.0, 0.0)
    # rejected below w_min
    assert oracle.interp(cal, m, 5.9, 5.9, oracle.BILINEAR, w_min=0.5)[:2] == (0.0, 0.0)
    # taps outside the frame count as bad: at x = -0.25 a quarter of the mass is off-frame
    v, w, _ = oracle.interp(cal, m, -0.25, 3.0, oracle.BILINEAR, w_min=0.5)
    assert abs(w - 0.75) < 1e-15 and abs(v - cal[3, 0]) < 1e-9
    # fully outside
    assert oracle.interp(cal, m, -5.0, -5.0, oracle.BILINEAR)[:2] == (0.0, 0.0)
    # outputs are never NaN/Inf
    for x, y in [(-0.5, -0.5), (31.5, 23.5), (31.0, 23.0), (0.0, 0.0)]:
        for k in (oracle.BILINEAR, oracle.LANCZOS3):
            v, w, _ = oracle.interp(cal, m, x, y, k)
            assert math.isfinite(v) and math.isfinite(w)


def test_ambiguity_flag():
    cal, m = _img()
    m[6, 6] = 0
    # near an integer x with a bad tap entering the neighbouring cell's tap set -> flagged
    assert oracle.interp(cal, m, 5.00001, 5.5, oracle.BILINEAR)[2] == 1
    assert oracle.interp(cal, m, 6.99999, 6.5, oracle.BILINEAR)[2] == 1
    # far from integers -> not flagged even next to the bad pixel
    assert oracle.interp(cal, m, 5.3, 5.5, oracle.BILINEAR)[2] == 0
    # near an integer but all taps good -> not flagged (the interpolant is continuous there)
    assert oracle.interp(cal, m, 15.00001, 15.5, oracle.BILINEAR)[2] == 0
    # |w - w_min| < 1e-4 -> flagged
    assert oracle.interp(cal, m, 5.5, 5.5, oracle.BILINEAR, w_min=0.75)[2] == 1


def test_o7_coadd_closed_form():
    tiles = np.array([3, 7, 8], dtype=np.int64)
    ppt = 4
    s = np.zeros(12)
    ws = np.zeros(12)
    idx = np.array([3 * 4 + 1, 7 * 4 + 0, 8 * 4 + 3, 5 * 4 + 2, 3 * 4 + 1], dtype=np.int64)
    val = np.array([10.0, 20.0, 30.0, 40.0, 50.0])
    wt = np.array([1.0, 0.5, 0.25, 1.0, 0.5])
    skipped = oracle.coadd_accumulate(tiles, ppt, s, ws, idx, val, wt)
    assert skipped == 1
    exp_s = np.zeros(12)
    exp_w = np.zeros(12)
    exp_s[1] = 10 + 25
    exp_w[1] = 1.5
    exp_s[4] = 10
    exp_w[4] = 0.5
    exp_s[11] = 7.5
    exp_w[11] = 0.25
    assert np.array_equal(s, exp_s) and np.array_equal(ws, exp_w)
