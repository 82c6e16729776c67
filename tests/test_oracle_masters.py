"""Pins of oracle/masters.py: the pre-fused variant against the DEFINITION of calibration (the C
oracle's orc_calibrate, O1), closed forms, mask logic, and the storage-precision bounds that decide which formats meet
north_star's 1e-3 ADU + 1e-5 relative."""
import numpy as np
import pytest

import oracle
import synth
from oracle import masters as om


@pytest.fixture(scope="module")
def fr():
    return synth.inject_defects(synth.config0())


def test_unrounded_prefused_equals_the_definition(fr):
    """(raw - (bias + dark t)) * (1/flat) with unrounded masters is O1 up to fp64 rounding; the masks are identical
    (saturated block, bad column, flat < flat_min patch, NaN flat)."""
    cal, mask = oracle.calibrate_frame(fr)
    off, gain = om.prepare_masters(fr.bias, fr.dark, fr.flat, fr.bpm, fr.t_exp, fr.flat_min, "f64")
    cal2, mask2 = om.calibrate_prefused(fr.raw, off, gain, fr.sat_adu)
    assert np.array_equal(mask, mask2) and 0 < mask.sum() < mask.size
    assert np.all(np.abs(cal2 - cal) <= 4e-16 * (np.abs(cal) + 1100.0))


def test_closed_form_constant_masters():
    raw = np.array([[1000, 1234, 65535, 0]], dtype=np.uint16)
    bias = np.full((1, 4), 1000.0, np.float32); dark = np.full((1, 4), 0.5, np.float32); flat = np.full((1, 4), 0.8, np.float32)
    off, gain = om.prepare_masters(bias, dark, flat, None, 30.0, 0.1, "f64")
    assert np.all(off == 1015.0) and np.allclose(gain, 1.0 / float(np.float32(0.8)), rtol=1e-15)
    cal, mask = om.calibrate_prefused(raw, off, gain, 65535)
    assert mask.tolist() == [[1, 1, 0, 1]]
    assert np.allclose(cal[0, [0, 1, 3]], np.array([-15.0, 219.0, -1015.0]) / float(np.float32(0.8)), rtol=1e-15)
    assert cal[0, 2] == 0.0


def test_invalid_pixels_fold_into_the_gain():
    bias = np.array([[1000, 1000, np.inf, 1000, 1000, 1000]], np.float32)
    dark = np.array([[0, 0, 0, np.nan, 0, 0]], np.float32)
    flat = np.array([[1.0, 0.05, 1.0, 1.0, np.nan, 1.0]], np.float32)
    bpm = np.array([[0, 0, 0, 0, 0, 7]], np.uint8)
    for fmt in ("f64", "f32", "f16"):
        off, gain = om.prepare_masters(bias, dark, flat, bpm, 1.0, 0.1, fmt)
        assert np.isnan(gain[0]).tolist() == [False, True, True, True, True, True], fmt
        assert np.all(np.isfinite(off))
        cal, mask = om.calibrate_prefused(np.full((1, 6), 1500, np.uint16), off, gain)
        assert mask[0].tolist() == [1, 0, 0, 0, 0, 0] and np.all(cal[0, 1:] == 0)
    # flat exactly at flat_min is valid (>=); just below is not
    fm = np.float32(0.1)
    off, gain = om.prepare_masters(np.zeros((1, 2), np.float32), np.zeros((1, 2), np.float32),
                                   np.array([[fm, np.nextafter(fm, np.float32(0))]], np.float32), None, 1.0, 0.1, "f32")
    assert np.isnan(gain[0]).tolist() == [False, True]


def test_binary16_storage_limits():
    """An offset beyond the binary16 range cannot be stored: the pixel becomes invalid rather than wrong."""
    bias = np.array([[1000.0, 70000.0]], np.float32)
    z = np.zeros((1, 2), np.float32); one = np.ones((1, 2), np.float32)
    off, gain = om.prepare_masters(bias, z, one, None, 1.0, 0.1, "f16")
    assert off.dtype == np.float16 and np.isnan(gain[0]).tolist() == [False, True]
    # round to nearest even at the binary16 grid: 1000.25 -> 1000.0 (ulp 0.5 in [512, 1024)), 1000.75 -> 1001.0 (tie -> even)
    off, _ = om.prepare_masters(np.array([[1000.25, 1000.75, 2049.0]], np.float32), np.zeros((1, 3), np.float32),
                                np.ones((1, 3), np.float32), None, 1.0, 0.1, "f16")
    assert off[0].astype(np.float64).tolist() == [1000.0, 1001.0, 2048.0]


@pytest.mark.parametrize("fmt,meets", [("f32", True), ("f16", False)])
def test_storage_precision_against_the_north_star_tolerance(fr, fmt, meets):
    """float32 masters keep every pixel of config 0 inside 1e-3 ADU + 1e-5 relative of the definition (and inside the
    analytic bound u (|offset| |gain| + |cal|)); binary16 masters do not: their error reaches the bound's order
    (0.15 ADU from rounding the 1000.15-ADU offset to the 0.5-ADU binary16 grid, up to 0.1 ADU more from the gain's
    2^-11 relative rounding on a 200-ADU sky) -- a median of tens of times the tolerance, 90 x at worst.  This is the statement DESIGN.md section 12 makes."""
    cal, mask = oracle.calibrate_frame(fr)
    off, gain = om.prepare_masters(fr.bias, fr.dark, fr.flat, fr.bpm, fr.t_exp, fr.flat_min, fmt)
    cal2, mask2 = om.calibrate_prefused(fr.raw, off, gain, fr.sat_adu)
    assert np.array_equal(mask, mask2)
    good = mask == 1
    err = np.abs(cal2 - cal)[good]
    bound = om.storage_error_bound(off.astype(np.float64), gain.astype(np.float64), cal, fmt)[good]
    assert np.all(err <= bound)
    tol = 1e-3 + 1e-5 * np.abs(cal[good])
    if meets:
        assert (err / tol).max() < 0.2
    else:
        assert (err / tol).max() > 50 and np.median(err / tol) > 10
