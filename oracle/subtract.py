"""Double-precision CPU oracle for direct image subtraction per tile.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.  Never imported
by paper_2207_14304_b200/.  Plain numpy, fp64, one tile at a time; no blocking or reordering beyond the definitions.

What the paper fixes: "Transient detection is performed using image subtraction in the reprojected HEALPix image
segments, leveraging long-term coadds as reference frames" (sec. 5.2); two algorithms, of which "the
direct image subtraction method ... for real-time operation in 1-second cadence data" is this row (ZOGY is the other);
it runs per tile, "parallelizing the direct subtraction at the segment level", 20 ms per tile on the CPU, "a GPU
implementation is in development" (Table 2); Figure 3 shows a science segment, a
reference, the difference and an injected transient "with a 5-sigma peak significance".  The method itself is in ref
[17], which is not in the container: every formula below is a DESIGN.md section 13 reading (R-X1 .. R-X8), the plain
scheme those sentences describe (reference = coadd, photometric match, difference, noise, thresholded local maxima).

Data layout: the tile-dense HEALPix layout of argus_coadd: sorted NSIDE_tile tile ids, each owning
ppt = (nside / nside_tile)^2 consecutive slots in NESTED order.  Both images are (sum, wsum) pairs as
argus_resample_coadd writes them: image = sum / wsum.

  R-X1 images     s = sci_sum / sci_wsum where sci_wsum >= sci_wmin, r = ref_sum / ref_wsum where ref_wsum >= ref_wmin;
                  a pixel is VALID iff both hold.
  R-X2 match      per tile, over its valid pixels: none: alpha = 1, beta = 0.  affine: least squares of s ~ alpha r +
                  beta (transparency and sky level differ between a 1 s exposure and a long coadd):
                  alpha = (n Srs - Sr Ss) / (n Srr - Sr^2), beta = (Ss - alpha Sr) / n; with fewer than n_min valid
                  pixels or a reference without structure -- n Srr - Sr^2 <= 1e-10 n Srr, i.e. variance(r) <= 1e-10
                  mean(r^2): constant up to rounding, where the slope is undetermined -- alpha = 1, beta = (Ss - Sr) / n
                  (0 if n = 0).
  R-X3 difference d = s - (alpha r + beta) at valid pixels, 0 elsewhere.
  R-X4 noise      m = alpha r + beta (the reference's prediction of the science pixel);
                  sigma^2 = (read_noise^2 + max(m, 0) / gain) * (1 / sci_wsum + alpha^2 / ref_wsum)
                  (one exposure's variance at level m, CCD equation in ADU; the averages of sci_wsum and ref_wsum
                  unit-weight exposures carry 1/wsum of it; the reference term is scaled by alpha^2).
  R-X5 S = d / sigma at valid pixels, 0 elsewhere.
  R-X6 detection  a valid pixel p is a candidate iff S_p > k, and S_p is the maximum over its valid 8-neighbours IN THE
                  TILE's (ix, iy) grid (tiles are independent; ix = even bits, iy = odd bits of the
                  in-tile nested index): S_p > S_q for neighbours q with a smaller nested index, S_p >= S_q for larger.
  R-X7 record     nested pixel index at nside, S_p, d_p, flux = sum of d over the valid pixels of the 3 x 3 window,
                  sigma_p, rank of the tile in the layout.
  R-X8 order      ascending nested pixel index.
"""
from __future__ import annotations

import numpy as np

MATCH_NONE, MATCH_AFFINE = 0, 1
FLAT_REFERENCE = 1e-10   # R-X2: variance(r) / mean(r^2) below which the reference has no structure to fit a slope to


def deinterleave(q, bits):
    """(ix, iy) of the in-tile nested index q: ix = even bits, iy = odd bits (HEALPix nested scheme, ref [10])."""
    q = np.asarray(q, dtype=np.int64)
    ix = np.zeros_like(q)
    iy = np.zeros_like(q)
    for b in range(bits):
        ix |= ((q >> (2 * b)) & 1) << b
        iy |= ((q >> (2 * b + 1)) & 1) << b
    return ix, iy


def tile_to_grid(a, side):
    """Nested-order tile array [side*side] -> [iy][ix] image."""
    bits = side.bit_length() - 1
    ix, iy = deinterleave(np.arange(side * side), bits)
    g = np.empty((side, side), dtype=np.asarray(a).dtype)
    g[iy, ix] = a
    return g


def grid_to_tile(g):
    side = g.shape[0]
    bits = side.bit_length() - 1
    ix, iy = deinterleave(np.arange(side * side), bits)
    return g[iy, ix]


def match_tile(s, r, valid, match=MATCH_AFFINE, n_min=16):
    """R-X2 on one tile.  Returns (alpha, beta, n_valid)."""
    n = int(valid.sum())
    if n == 0:
        return 1.0, 0.0, 0
    sv, rv = s[valid], r[valid]
    Ss, Sr = sv.sum(), rv.sum()
    if match == MATCH_NONE:
        return 1.0, 0.0, n
    Srr = (rv * rv).sum()
    den = n * Srr - Sr * Sr
    if n < n_min or not den > FLAT_REFERENCE * n * Srr:
        return 1.0, (Ss - Sr) / n, n
    alpha = (n * (rv * sv).sum() - Sr * Ss) / den
    return alpha, (Ss - alpha * Sr) / n, n


_NEIGH = [(-1, -1), (-1, 0), (-1, 1), (0, -1), (0, 1), (1, -1), (1, 0), (1, 1)]   # (diy, dix)


def subtract_tiles(tiles, ppt, nside, sci_sum, sci_wsum, ref_sum, ref_wsum, match=MATCH_AFFINE, n_min=16, sci_wmin=0.5,
                   ref_wmin=0.5, read_noise=1.7, gain=1.0, k_sigma=5.0, slack=0.0):
    """R-X1 .. R-X8.  Returns dict(diff, sig, alpha, beta, n_valid, cat) where cat is a dict of arrays over the
    candidates in ascending nested order: pixel, sig, diff, flux, noise, tile_rank, plus the decision margins m_thr =
    S - k and m_max = min over valid neighbours of (S_p - S_q) and `strict`; slack > 0 also lists the near misses."""
    tiles = np.asarray(tiles, dtype=np.int64)
    side = int(round(np.sqrt(ppt)))
    assert side * side == ppt
    n_tiles = len(tiles)
    f = lambda a: np.asarray(a, dtype=np.float64).reshape(n_tiles, ppt)
    ss, sw, rs, rw = f(sci_sum), f(sci_wsum), f(ref_sum), f(ref_wsum)
    diff = np.zeros((n_tiles, ppt)); sig = np.zeros((n_tiles, ppt))
    alpha = np.ones(n_tiles); beta = np.zeros(n_tiles); n_valid = np.zeros(n_tiles, dtype=np.int64)
    cat = {k: [] for k in ("pixel", "sig", "diff", "flux", "noise", "tile_rank", "m_thr", "m_max", "strict")}
    bits = side.bit_length() - 1
    qix, qiy = deinterleave(np.arange(ppt), bits)
    for t in range(n_tiles):
        valid = (sw[t] >= sci_wmin) & (rw[t] >= ref_wmin)
        with np.errstate(all="ignore"):
            s = np.where(valid, ss[t] / np.where(valid, sw[t], 1.0), 0.0)
            r = np.where(valid, rs[t] / np.where(valid, rw[t], 1.0), 0.0)
        a, b, n = match_tile(s, r, valid, match, n_min)
        alpha[t], beta[t], n_valid[t] = a, b, n
        m = a * r + b
        d = np.where(valid, s - m, 0.0)
        with np.errstate(all="ignore"):
            var = (read_noise ** 2 + np.maximum(m, 0.0) / gain) * (1.0 / np.where(valid, sw[t], 1.0) + a * a / np.where(valid, rw[t], 1.0))
        sigma = np.sqrt(var)
        S = np.where(valid, d / np.where(valid, sigma, 1.0), 0.0)
        diff[t], sig[t] = d, S
        # detection on the tile's (iy, ix) grid
        Sg = np.full((side + 2, side + 2), -np.inf)
        Sg[1:-1, 1:-1] = tile_to_grid(np.where(valid, S, -np.inf), side)
        dg = np.zeros((side + 2, side + 2)); dg[1:-1, 1:-1] = tile_to_grid(d, side)
        vg = np.zeros((side + 2, side + 2), dtype=bool); vg[1:-1, 1:-1] = tile_to_grid(valid, side)
        qg = np.full((side + 2, side + 2), -1, dtype=np.int64); qg[1:-1, 1:-1] = tile_to_grid(np.arange(ppt), side)
        C = Sg[1:-1, 1:-1]
        m_max = np.full((side, side), np.inf)
        strict = np.ones((side, side), dtype=bool)
        for diy, dix in _NEIGH:
            Q = Sg[1 + diy:1 + diy + side, 1 + dix:1 + dix + side]
            qq = qg[1 + diy:1 + diy + side, 1 + dix:1 + dix + side]
            with np.errstate(invalid="ignore"):
                dd = np.where(np.isfinite(Q), C - Q, np.inf)
            m_max = np.minimum(m_max, dd)
            before = qq < qg[1:-1, 1:-1]              # neighbour has the smaller nested index: p must beat it strictly
            strict &= np.where(before, dd > 0, dd >= 0)
        m_thr = np.where(vg[1:-1, 1:-1], C - k_sigma, -np.inf)
        cand = ((m_thr > -slack) & (m_max > -slack)) if slack > 0 else ((m_thr > 0) & strict)
        iy, ix = np.nonzero(cand)
        q = qg[1 + iy, 1 + ix]
        o = np.argsort(q)
        iy, ix, q = iy[o], ix[o], q[o]
        flux = np.zeros(len(q))
        for diy in (-1, 0, 1):
            for dix in (-1, 0, 1):
                flux += np.where(vg[1 + iy + diy, 1 + ix + dix], dg[1 + iy + diy, 1 + ix + dix], 0.0)
        cat["pixel"].append(tiles[t] * ppt + q)
        cat["sig"].append(S[q]); cat["diff"].append(d[q]); cat["flux"].append(flux); cat["noise"].append(sigma[q])
        cat["tile_rank"].append(np.full(len(q), t, dtype=np.int64))
        cat["m_thr"].append(m_thr[iy, ix]); cat["m_max"].append(m_max[iy, ix])
        cat["strict"].append((m_thr[iy, ix] > 0) & strict[iy, ix])
    cat = {k: (np.concatenate(v) if v else np.zeros(0)) for k, v in cat.items()}
    return dict(diff=diff.reshape(-1), sig=sig.reshape(-1), alpha=alpha, beta=beta, n_valid=n_valid, cat=cat)
