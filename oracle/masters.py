"""Double-precision CPU oracle for pre-fused / reduced-precision calibration masters (DESIGN.md
section 12).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.  Never imported
by paper_2207_14304_b200/.  Plain numpy, fp64.

What the paper fixes: calibration = "dark subtraction, flat fielding, masking of bad pixels" (Table 2
:192), with the masters uploaded once "at the start of each pointing" and resident on the GPU.
Everything that depends only on the masters and the exposure time can therefore be formed once per pointing.  The
DEFINITION of the calibrated pixel stays O1 of SURVEY.md 8(c), cal = (raw - bias - dark * t_exp) / flat
(oracle/argus_oracle.c: orc_calibrate); this module states what the pre-fused variant stores and computes, so that its
deviation from the definition can be bounded and measured:

  R-M1 offset = bias + dark * t_exp                      (ADU; one number per pixel and exposure time)
  R-M2 gain   = 1 / flat where the pixel is valid, NaN where it is not: flat < flat_min or not finite, bias or dark
                not finite, bpm != 0 (the bad-pixel mask folds into the gain, "masking of bad pixels")
  R-M3 stored as float32 or as IEEE binary16 (round to nearest even; an offset beyond the binary16 range makes the
       pixel invalid)
  R-M4 cal = (raw - offset) * gain on the STORED values; masked iff raw >= sat_adu or gain is NaN
"""
from __future__ import annotations

import numpy as np

FORMATS = {"f64": np.float64, "f32": np.float32, "f16": np.float16}


def prepare_masters(bias, dark, flat, bpm, t_exp, flat_min=0.1, fmt="f32"):
    """R-M1 .. R-M3.  Returns (offset, gain) as arrays of the storage dtype (fmt "f64" = unrounded, for the pins)."""
    bias = np.asarray(bias, dtype=np.float64)
    dark = np.asarray(dark, dtype=np.float64)
    flat = np.asarray(flat, dtype=np.float64)
    t = float(np.float32(t_exp))                       # the C ABI passes t_exp as a float
    with np.errstate(all="ignore"):
        offset = bias + dark * t
        valid = (flat >= float(np.float32(flat_min))) & np.isfinite(flat) & np.isfinite(bias) & np.isfinite(dark)
        if bpm is not None:
            valid &= np.asarray(bpm) == 0
        gain = np.where(valid, 1.0 / np.where(valid, flat, 1.0), np.nan)
        dt = FORMATS[fmt]
        offset_s = offset.astype(dt)
        gain_s = gain.astype(dt)
        lost = valid & ~(np.isfinite(offset_s) & np.isfinite(gain_s))    # not representable in the storage format
        gain_s[lost] = np.nan
        offset_s[~np.isfinite(offset_s)] = 0
    return offset_s, gain_s


def calibrate_prefused(raw, offset, gain, sat_adu=65535):
    """R-M4 in fp64 on the stored masters.  Returns (cal float64 [H][W] with 0 where masked, mask uint8, 1 = good)."""
    raw = np.asarray(raw)
    off = np.asarray(offset).astype(np.float64)
    g = np.asarray(gain).astype(np.float64)
    with np.errstate(all="ignore"):
        cal = (raw.astype(np.float64) - off) * g
    good = (raw < sat_adu) & np.isfinite(cal)
    return np.where(good, cal, 0.0), good.astype(np.uint8)


def storage_error_bound(offset, gain, cal, fmt):
    """|cal_stored - cal_definition| <= u (|offset| |gain| + |cal|) (1 + u) for storage unit roundoff u (2^-24 float32,
    2^-11 binary16): offset and gain each carry a relative rounding error of at most u."""
    u = {"f32": 2.0 ** -24, "f16": 2.0 ** -11, "f64": 2.0 ** -53}[fmt]
    return u * (np.abs(offset) * np.abs(gain) + np.abs(cal)) * (1.0 + 2 * u) + 4 * np.finfo(np.float64).eps * np.abs(cal)
