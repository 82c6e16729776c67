"""Double-precision CPU oracle for the segment products.

TEST INFRASTRUCTURE ONLY: imported by tests/ and bench.py's cpu_baseline leg.  Never imported by
paper_2207_14304_b200/.  Plain numpy, fp64 sums; no blocking or reordering beyond the definitions below.

What the paper fixes (everything else is a DESIGN.md section 10 reading):
  * PAPER.md:145  segment images are stored as 16-bit float data;
  * PAPER.md:149  "stamping": minipix segments of each image tile, at the higher HEALPix level NSIDE = 16384,
                  that contain no science target are set to zero;
  * PAPER.md:73, :149  low-resolution maps at 13.8 arcsec per pixel (10x the 1.38 arcsec detector scale).
In the nested scheme (ref [10]) the pixel p at nside = 2^k lies in the pixel p >> 2j at
nside / 2^j; at nside 2^17 a minipix (NSIDE 16384 = 2^14) is 4^3 = 64 consecutive nested indices, 12.9 arcsec
across: the HEALPix level nearest the paper's 13.8 arcsec, which is what the low-resolution map is built on
here (reading R-S3).

Functions
  minipix_of(idx, nside, nside_mini)        parent pixel at nside_mini (pinned against ang2pix(pix2ang))
  pack_f16(v)                               IEEE binary16 bits, round-to-nearest-even, finite values clamped to
                                            +-65504, NaN -> 0x7e00 (pinned against struct 'e' and hand values)
  raster_offset(local, side)                row-major position of an in-tile nested index (pinned against nest2xyf)
  segment_products(...)                     stamping + packing + low-resolution weighted means
"""
from __future__ import annotations

import numpy as np

F16_MAX = 65504.0


def _log2_exact(n):
    n = int(n)
    if n < 1 or n & (n - 1):
        raise ValueError("not a power of two: %r" % (n,))
    return n.bit_length() - 1


def minipix_of(idx, nside, nside_mini):
    """Parent of nested pixel idx (at nside) at resolution nside_mini <= nside: idx >> 2j, 2^j = nside/nside_mini."""
    j = _log2_exact(nside) - _log2_exact(nside_mini)
    if j < 0:
        raise ValueError("nside_mini > nside")
    return np.asarray(idx, dtype=np.int64) >> (2 * j)


def pack_f16(v):
    """float -> IEEE binary16 bit patterns (uint16).  Reading R-S2: finite values beyond the binary16 range
    are clamped to +-65504 (the files hold finite data only); NaN becomes the canonical quiet NaN 0x7e00."""
    v = np.asarray(v, dtype=np.float32)
    nan = np.isnan(v)
    c = np.clip(np.where(nan, np.float32(0), v), np.float32(-F16_MAX), np.float32(F16_MAX))
    bits = c.astype(np.float16).view(np.uint16).copy()   # numpy converts with round-to-nearest-even
    bits[nan] = 0x7E00
    return bits


def raster_offset(local, side):
    """Row-major position iy * side + ix inside a tile of side x side pixels of the pixel whose in-tile nested
    index is `local` (ref [10]: ix = the even bits of the nested index, iy = the odd bits; reading R-S5: x runs
    fastest).  Written out bit by bit."""
    local = np.asarray(local, dtype=np.int64)
    nb = _log2_exact(side)
    ix = np.zeros_like(local)
    iy = np.zeros_like(local)
    for b in range(nb):
        ix |= ((local >> (2 * b)) & 1) << b
        iy |= ((local >> (2 * b + 1)) & 1) << b
    return iy * side + ix


def segment_products(idx, value, weight, nside, nside_mini, targets, layout_tiles=None, nside_tile=None, raster=False):
    """idx: ascending unique nested pixels at nside (a footprint); value, weight: the resampled frame on them.
    targets: minipix ids (at nside_mini) that hold a science target (any order, duplicates allowed).

    Returns a dict:
      mini_id      ascending ids of the minipix that own at least one footprint pixel
      mini_keep    1 where mini_id is in targets
      mini_weight  sum of weight over the minipix' footprint pixels                      (fp64)
      mini_value   sum(weight * value) / sum(weight), 0 where the sum of weights is 0     (fp64)
      seg16        binary16 bits of value where the pixel's minipix is kept, of 0 elsewhere; element i <-> idx[i]
      dense16      (when layout_tiles is given) seg16 scattered to slot(p) = rank(p / ppt) * ppt + p % ppt with
                   ppt = (nside / nside_tile)^2, zeros elsewhere; pixels whose tile is absent are dropped;
                   raster=True: each tile is a row-major image, p % ppt replaced by raster_offset(p % ppt)
    """
    idx = np.asarray(idx, dtype=np.int64)
    value = np.asarray(value, dtype=np.float64)
    weight = np.asarray(weight, dtype=np.float64)
    m = minipix_of(idx, nside, nside_mini)
    mini_id, inv = np.unique(m, return_inverse=True)
    n_mini = mini_id.size
    tset = np.unique(np.asarray(targets, dtype=np.int64))
    mini_keep = np.isin(mini_id, tset).astype(np.uint8)
    sw = np.bincount(inv, weights=weight, minlength=n_mini)
    swv = np.bincount(inv, weights=weight * value, minlength=n_mini)
    with np.errstate(invalid="ignore", divide="ignore"):
        mini_value = np.where(sw != 0, swv / np.where(sw != 0, sw, 1.0), 0.0)
    keep_px = mini_keep[inv].astype(bool) if n_mini else np.zeros(0, bool)
    seg16 = pack_f16(np.where(keep_px, value.astype(np.float32), np.float32(0)))
    out = dict(mini_id=mini_id, mini_keep=mini_keep, mini_weight=sw, mini_value=mini_value, seg16=seg16)
    if layout_tiles is not None:
        tiles = np.asarray(layout_tiles, dtype=np.int64)
        kk = _log2_exact(nside) - _log2_exact(nside_tile)
        ppt = 1 << (2 * kk)
        dense = np.zeros(tiles.size * ppt, dtype=np.uint16)
        key = idx >> (2 * kk)
        pos = np.searchsorted(tiles, key)
        ok = (pos < tiles.size)
        ok[ok] &= tiles[pos[ok]] == key[ok]
        local = idx[ok] & (ppt - 1)
        dense[pos[ok] * ppt + (raster_offset(local, 1 << kk) if raster else local)] = seg16[ok]
        out["dense16"] = dense
    return out
