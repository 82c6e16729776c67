"""Pin P6 for the oracle's sky->pixel mapping (O4): the textbook forward gnomonic deprojection
(pixel -> sky, closed form, written here independently) composed with the oracle is the identity;
special directions; SIP polynomial against mpmath at 50 digits."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle
import synth

D2R = math.pi / 180.0


def forward_tan(wcs, x, y):
    """Textbook gnomonic deprojection about (a0, d0) (no SIP): pixel -> (alpha, delta)."""
    a0, d0 = wcs.crval[0] * D2R, wcs.crval[1] * D2R
    U, V = x - wcs.crpix[0], y - wcs.crpix[1]
    xi = (wcs.cd[0][0] * U + wcs.cd[0][1] * V) * D2R
    eta = (wcs.cd[1][0] * U + wcs.cd[1][1] * V) * D2R
    alpha = a0 + math.atan2(xi, math.cos(d0) - eta * math.sin(d0))
    delta = math.atan2((math.sin(d0) + eta * math.cos(d0)),
                       math.hypot(xi, math.cos(d0) - eta * math.sin(d0)))
    return alpha, delta


@pytest.mark.parametrize("crval,rot", [((30.0, 20.0), 0.3), ((0.0, -20.0), 45.0), ((359.9, 72.0), -1.0),
                                       ((123.0, 89.9), 10.0), ((200.0, -60.0), 170.0), ((45.0, 0.0), 0.0)])
def test_p6_forward_inverse_roundtrip(crval, rot):
    W, H = 9576, 6388
    wcs = synth.make_wcs(crval, ((W - 1) / 2.0, (H - 1) / 2.0), rot)
    rng = np.random.default_rng(5)
    pts = [(-0.5, -0.5), (W - 0.5, -0.5), (-0.5, H - 0.5), (W - 0.5, H - 0.5)]
    pts += [(rng.uniform(-0.5, W - 0.5), rng.uniform(-0.5, H - 0.5)) for _ in range(400)]
    for x, y in pts:
        a, d = forward_tan(wcs, x, y)
        xo, yo, cosc = oracle.sky2pix(wcs, a, d)
        assert cosc > 0.99
        assert abs(xo - x) < 1e-9 and abs(yo - y) < 1e-9


def test_p6_special_directions():
    wcs = synth.make_wcs((30.0, 20.0), (255.5, 255.5), 0.0)
    s = synth.PIXEL_SCALE_DEG * D2R
    # CRVAL maps to CRPIX exactly
    x, y, c = oracle.sky2pix(wcs, 30.0 * D2R, 20.0 * D2R)
    assert (x, y, c) == (255.5, 255.5, 1.0) or (abs(x - 255.5) < 1e-12 and abs(y - 255.5) < 1e-12 and abs(c - 1) < 1e-15)
    # a point rho due north: eta = tan(rho), xi = 0 -> y = crpix + tan(rho)/s (north-up at rotation 0)
    rho = 1.3 * D2R
    x, y, c = oracle.sky2pix(wcs, 30.0 * D2R, 20.0 * D2R + rho)
    assert abs(x - 255.5) < 1e-9
    assert abs((y - 255.5) - math.tan(rho) / s) < 1e-8
    assert abs(c - math.cos(rho)) < 1e-15
    # a point to the east (larger alpha) lands at smaller x (east-left)
    x, y, c = oracle.sky2pix(wcs, 30.5 * D2R, 20.0 * D2R)
    assert x < 255.5 - 100
    # on the great circle through CRVAL perpendicular to the meridian y barely changes sign: eta > 0 small
    assert 0 < y - 255.5 < 20
    # antipode and beyond 90 degrees: rejected (cos c <= 0)
    x, y, c = oracle.sky2pix(wcs, 210.0 * D2R, -20.0 * D2R)
    assert c < 0 and math.isnan(x)


def test_p6_rotation_sense():
    """CD = s[[-cos r, sin r],[sin r, cos r]]: at r = 90 deg north maps to +x."""
    wcs = synth.make_wcs((10.0, 0.0), (0.0, 0.0), 90.0)
    x, y, _ = oracle.sky2pix(wcs, 10.0 * D2R, 0.5 * D2R)
    assert x > 1000 and abs(y) < 1e-6


def test_p6_sip_zero_equals_tan():
    base = synth.make_wcs((30.0, 20.0), (100.0, 80.0), 12.0)
    sip0 = synth.make_wcs((30.0, 20.0), (100.0, 80.0), 12.0, sip=(3, np.zeros(36), np.zeros(36)))
    rng = np.random.default_rng(2)
    for _ in range(100):
        a, d = (30 + rng.uniform(-1, 1)) * D2R, (20 + rng.uniform(-1, 1)) * D2R
        assert oracle.sky2pix(base, a, d) == oracle.sky2pix(sip0, a, d)


def test_p6_sip_polynomial_mpmath():
    """Whole O4 chain recomputed with mpmath at 50 digits in VECTOR form (dot products with the
    east/north/normal basis at CRVAL), including the AP/BP polynomial with [p*6+q] indexing."""
    mp.mp.dps = 50
    rng = np.random.default_rng(11)
    sip = synth.make_sip(rng, 5, 4788.0)
    # make the coefficients asymmetric and large enough that an index transposition is visible
    sip[1][1 * 6 + 2] = 3e-10
    sip[1][2 * 6 + 1] = -7e-10
    sip[2][0 * 6 + 2] = 2e-6
    sip[2][2 * 6 + 0] = -1e-6
    wcs = synth.make_wcs((137.5, 55.0), (4787.5, 3193.5), 0.7, sip=sip)
    a0, d0 = mp.mpf(wcs.crval[0]) * mp.pi / 180, mp.mpf(wcs.crval[1]) * mp.pi / 180
    e_r = mp.matrix([mp.cos(d0) * mp.cos(a0), mp.cos(d0) * mp.sin(a0), mp.sin(d0)])
    e_e = mp.matrix([-mp.sin(a0), mp.cos(a0), 0])
    e_n = mp.matrix([-mp.sin(d0) * mp.cos(a0), -mp.sin(d0) * mp.sin(a0), mp.cos(d0)])
    cd = mp.matrix([[mp.mpf(wcs.cd[0][0]), mp.mpf(wcs.cd[0][1])], [mp.mpf(wcs.cd[1][0]), mp.mpf(wcs.cd[1][1])]])
    cdi = cd ** -1
    for _ in range(50):
        a = (wcs.crval[0] + rng.uniform(-2.5, 2.5)) * D2R
        d = (wcs.crval[1] + rng.uniform(-1.5, 1.5)) * D2R
        am, dm = mp.mpf(a), mp.mpf(d)
        v = mp.matrix([mp.cos(dm) * mp.cos(am), mp.cos(dm) * mp.sin(am), mp.sin(dm)])
        c = (v.T * e_r)[0]
        xi = (v.T * e_e)[0] / c * 180 / mp.pi
        eta = (v.T * e_n)[0] / c * 180 / mp.pi
        UV = cdi * mp.matrix([xi, eta])
        U, V = UV[0], UV[1]
        fu = sum(mp.mpf(float(wcs.ap[p * 6 + q])) * U ** p * V ** q for p in range(6) for q in range(6) if p + q <= 5)
        fv = sum(mp.mpf(float(wcs.bp[p * 6 + q])) * U ** p * V ** q for p in range(6) for q in range(6) if p + q <= 5)
        xm, ym = U + fu + mp.mpf(wcs.crpix[0]), V + fv + mp.mpf(wcs.crpix[1])
        x, y, cc = oracle.sky2pix(wcs, a, d)
        assert abs(x - float(xm)) < 2e-9 and abs(y - float(ym)) < 2e-9
        assert abs(cc - float(c)) < 1e-15


def test_rho_max_reading():
    wcs = synth.make_wcs((30.0, 20.0), (4787.5, 3193.5), 0.3)
    c = oracle.cos_rho_max(wcs, 9576, 6388)
    rho = math.degrees(math.acos(c))
    assert abs(rho - 2.76) < 0.01  # config 1 => ~2.76 deg
    # every frame corner lies inside the cone with margin
    for x, y in [(-0.5, -0.5), (9575.5, 6387.5), (-0.5, 6387.5), (9575.5, -0.5)]:
        a, d = forward_tan(wcs, x, y)
        assert oracle.sky2pix(wcs, a, d)[2] > c + 1e-4
