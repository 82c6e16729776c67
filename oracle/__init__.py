"""ctypes wrapper over the double-precision CPU oracle (oracle/argus_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_2207_14304_b200/.
Argument marshalling only; all arithmetic lives in argus_oracle.c (see its header for citations).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

BILINEAR, LANCZOS3 = 0, 1
KERNELS = {"bilinear": BILINEAR, "lanczos3": LANCZOS3}

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        i64, f64, vp, ci = C.c_int64, C.c_double, C.c_void_p, C.c_int
        L.orc_max_threads.restype = ci
        L.orc_set_threads.argtypes = [ci]
        L.orc_calibrate.argtypes = [vp, vp, vp, vp, vp, i64, i64, f64, ci, f64, vp, vp]
        L.orc_nest2xyf.argtypes = [i64, i64, vp, vp, vp]
        L.orc_xyf2nest.argtypes = [i64, ci, i64, i64]
        L.orc_xyf2nest.restype = i64
        L.orc_pix2ang_nest.argtypes = [i64, i64, vp, vp]
        L.orc_ang2pix_nest.argtypes = [i64, f64, f64]
        L.orc_ang2pix_nest.restype = i64
        L.orc_sky2pix.argtypes = [vp, f64, f64, vp, vp]
        L.orc_sky2pix.restype = f64
        L.orc_cos_rho_max.argtypes = [vp, i64, i64]
        L.orc_cos_rho_max.restype = f64
        L.orc_pix2xy_many.argtypes = [vp, i64, vp, i64, vp, vp, vp]
        L.orc_member.argtypes = [vp, i64, i64, i64, i64, f64, vp]
        L.orc_member.restype = ci
        L.orc_footprint.argtypes = [vp, i64, i64, i64, i64, vp, i64, vp]
        L.orc_footprint.restype = i64
        L.orc_interp.argtypes = [vp, vp, i64, i64, f64, f64, ci, f64, vp, vp, vp]
        L.orc_resample.argtypes = [vp, vp, i64, i64, vp, i64, ci, f64, vp, i64, vp, vp, vp, vp, vp]
        L.orc_coadd_accumulate.argtypes = [vp, i64, i64, vp, vp, vp, vp, vp, i64]
        L.orc_coadd_accumulate.restype = i64
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _wcs(w) -> np.ndarray:
    a = w.as_array() if hasattr(w, "as_array") else np.asarray(w, dtype=np.float64)
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == (81,)
    return a


def max_threads() -> int:
    return int(lib().orc_max_threads())


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def calibrate(raw, bias, dark, flat, bpm, t_exp, sat_adu=65535, flat_min=0.1):
    """O1.  Returns (cal float64 [H][W], mask uint8 [H][W], 1 = good)."""
    H, W = raw.shape
    raw = np.ascontiguousarray(raw, dtype=np.uint16)
    bias = np.ascontiguousarray(bias, dtype=np.float32)
    dark = np.ascontiguousarray(dark, dtype=np.float32)
    flat = np.ascontiguousarray(flat, dtype=np.float32)
    if bpm is not None:
        bpm = np.ascontiguousarray(bpm, dtype=np.uint8)
    cal = np.empty((H, W), dtype=np.float64)
    mask = np.empty((H, W), dtype=np.uint8)
    lib().orc_calibrate(_p(raw), _p(bias), _p(dark), _p(flat), _p(bpm), W, H, float(t_exp), int(sat_adu),
                        float(flat_min), _p(cal), _p(mask))
    return cal, mask


def calibrate_frame(fr):
    return calibrate(fr.raw, fr.bias, fr.dark, fr.flat, fr.bpm, fr.t_exp, fr.sat_adu, fr.flat_min)


def nest2xyf(nside, p):
    f = C.c_int()
    ix, iy = C.c_int64(), C.c_int64()
    lib().orc_nest2xyf(int(nside), int(p), C.byref(f), C.byref(ix), C.byref(iy))
    return f.value, ix.value, iy.value


def xyf2nest(nside, face, ix, iy):
    return int(lib().orc_xyf2nest(int(nside), int(face), int(ix), int(iy)))


def pix2ang(nside, p):
    """O3.  Returns (theta, phi) of the nested pixel centre."""
    th, ph = C.c_double(), C.c_double()
    lib().orc_pix2ang_nest(int(nside), int(p), C.byref(th), C.byref(ph))
    return th.value, ph.value


def ang2pix(nside, theta, phi):
    return int(lib().orc_ang2pix_nest(int(nside), float(theta), float(phi)))


def sky2pix(wcs, alpha, delta):
    """O4.  Returns (x, y, cos c)."""
    w = _wcs(wcs)
    x, y = C.c_double(), C.c_double()
    c = lib().orc_sky2pix(_p(w), float(alpha), float(delta), C.byref(x), C.byref(y))
    return x.value, y.value, float(c)


def cos_rho_max(wcs, W, H):
    w = _wcs(wcs)
    return float(lib().orc_cos_rho_max(_p(w), int(W), int(H)))


def pix2xy(wcs, nside, idx):
    """O2+O3+O4 for an array of nested indices.  Returns (x, y, cos c)."""
    w = _wcs(wcs)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    n = idx.size
    x = np.empty(n)
    y = np.empty(n)
    c = np.empty(n)
    lib().orc_pix2xy_many(_p(w), int(nside), _p(idx), n, _p(x), _p(y), _p(c))
    return x, y, c


def member(wcs, W, H, nside, p):
    """Exact footprint predicate for one pixel.  Returns (in_footprint, distance to domain border)."""
    w = _wcs(wcs)
    d = C.c_double()
    r = lib().orc_member(_p(w), int(W), int(H), int(nside), int(p), cos_rho_max(wcs, W, H), C.byref(d))
    return bool(r), d.value


def footprint(wcs, W, H, nside, split_nside=2048, count_only=False):
    """O5.  Returns (idx int64 ascending, min distance to the domain border in px)."""
    w = _wcs(wcs)
    dmin = C.c_double()
    n = lib().orc_footprint(_p(w), int(W), int(H), int(nside), int(split_nside), None, 0, C.byref(dmin))
    if count_only:
        return int(n), dmin.value
    idx = np.empty(int(n), dtype=np.int64)
    m = lib().orc_footprint(_p(w), int(W), int(H), int(nside), int(split_nside), _p(idx), int(n), C.byref(dmin))
    assert m == n
    return idx, dmin.value


def interp(cal, mask, x, y, kernel=BILINEAR, w_min=0.5):
    """O6 at one point.  Returns (value, weight, ambiguous flag)."""
    H, W = cal.shape
    cal = np.ascontiguousarray(cal, dtype=np.float64)
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    v, wt = C.c_double(), C.c_double()
    fl = C.c_uint8()
    lib().orc_interp(_p(cal), _p(mask), W, H, float(x), float(y), int(kernel), float(w_min), C.byref(v),
                     C.byref(wt), C.byref(fl))
    return v.value, wt.value, int(fl.value)


def resample(cal, mask, wcs, nside, idx, kernel=BILINEAR, w_min=0.5, return_xy=False):
    """O2..O6 for an index list.  Returns (value, weight, flag[, x, y])."""
    H, W = cal.shape
    w = _wcs(wcs)
    cal = np.ascontiguousarray(cal, dtype=np.float64)
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    n = idx.size
    value = np.empty(n)
    weight = np.empty(n)
    flag = np.empty(n, dtype=np.uint8)
    xs = np.empty(n) if return_xy else None
    ys = np.empty(n) if return_xy else None
    lib().orc_resample(_p(cal), _p(mask), W, H, _p(w), int(nside), int(kernel), float(w_min), _p(idx), n,
                       _p(value), _p(weight), _p(flag), _p(xs), _p(ys))
    if return_xy:
        return value, weight, flag, xs, ys
    return value, weight, flag


def coadd_accumulate(tiles, ppt, sum_, wsum, idx, value, weight):
    """O7 in place on float64 sum_/wsum.  Returns the number of skipped pixels."""
    tiles = np.ascontiguousarray(tiles, dtype=np.int64)
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    value = np.ascontiguousarray(value, dtype=np.float64)
    weight = np.ascontiguousarray(weight, dtype=np.float64)
    assert sum_.dtype == np.float64 and wsum.dtype == np.float64
    assert sum_.flags.c_contiguous and wsum.flags.c_contiguous
    return int(lib().orc_coadd_accumulate(_p(tiles), tiles.size, int(ppt), _p(sum_), _p(wsum), _p(idx),
                                          _p(value), _p(weight), idx.size))
