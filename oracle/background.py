"""Double-precision CPU oracle for the background map and source detection.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.  Never
imported by paper_2207_14304_b200/.  Plain numpy, fp64; no blocking or reordering beyond the definitions below.

What the paper fixes: the two GPU stages between calibration and resampling are a "Median-filtered background map"
and "Source detection" (Table 2; "source detection ... directly on the GPU"), the
per-camera calibration set holds "intermediate background and noise maps", and the detections leave
the GPU as a source catalogue.  The paper gives no formula; everything below is a DESIGN.md
section 11 reading (R-D1 .. R-D7), restating the textbook mesh-background / thresholded-local-maximum scheme.

Definitions (cal[H][W] calibrated ADU, mask[H][W] 1 = good; B = cell size; "median" of n values v_(0) <= ... <=
v_(n-1) is (v_((n-1)//2) + v_(n//2)) / 2):
  R-D1 cells      cell (gx, gy) = pixels [gx*B, min((gx+1)*B, W)) x [gy*B, min((gy+1)*B, H)); GX = ceil(W/B).
                  med = median of its good pixels, mad = median of |v - med|, sig = 1.4826 * mad; a cell with fewer
                  than n_min good pixels is invalid.
  R-D2 filter     bkg[gy][gx] = median of med over the VALID cells of the 3x3 cell neighbourhood (clipped to the grid,
                  the cell itself included); nse[gy][gx] likewise from sig; no valid cell: bkg = 0, nse = +inf.
  R-D3 per pixel  bilinear interpolation between cell centres cx = gx*B + (B-1)/2 (nominal, also for ragged cells),
                  clamped outside the outermost centres.
  R-D4 detect     s = cal - bkg(x, y); pixel p is a source iff mask = 1, s > k * nse(x, y), s > 0 and s is the
                  maximum over its good in-frame 8-neighbours q: s_p > s_q for q before p in raster order,
                  s_p >= s_q for q after p (of equal neighbours the raster-first one is the source).  A pixel touching an interpolation node with nse = +inf is never a source.
  R-D5 record     x, y, peak = s_p, flux = sum of s over the good in-frame pixels of the 3x3 window, centroid offsets
                  cx = sum(s * dx) / flux, cy = sum(s * dy) / flux (0 when flux <= 0), bkg and nse at p.
  R-D6 order      ascending raster index y * W + x (the paper hands the catalogue to CPU cross-matching, PAPER.md:135,
                  and states no order; raster order is the one that depends on nothing but the frame).
"""
from __future__ import annotations

import numpy as np

MAD_TO_SIGMA = 1.4826


def median_rule(v):
    """(v_((n-1)//2) + v_(n//2)) / 2 of the sorted values (R-D1); n >= 1."""
    s = np.sort(np.asarray(v, dtype=np.float64).ravel())
    n = s.size
    return 0.5 * (s[(n - 1) // 2] + s[n // 2])


def cell_stats(cal, mask, B=64, n_min=16):
    """R-D1.  Returns med[GY][GX], sig[GY][GX] (fp64; 0 where invalid), valid[GY][GX] (bool), n_good[GY][GX]."""
    cal = np.asarray(cal, dtype=np.float64)
    H, W = cal.shape
    GX, GY = -(-W // B), -(-H // B)
    med = np.zeros((GY, GX)); sig = np.zeros((GY, GX))
    valid = np.zeros((GY, GX), dtype=bool); n_good = np.zeros((GY, GX), dtype=np.int64)
    for gy in range(GY):
        for gx in range(GX):
            c = cal[gy * B:(gy + 1) * B, gx * B:(gx + 1) * B]
            m = np.asarray(mask[gy * B:(gy + 1) * B, gx * B:(gx + 1) * B]) != 0
            v = c[m]
            n_good[gy, gx] = v.size
            if v.size < max(1, n_min):
                continue
            valid[gy, gx] = True
            med[gy, gx] = median_rule(v)
            sig[gy, gx] = MAD_TO_SIGMA * median_rule(np.abs(v - med[gy, gx]))
    return med, sig, valid, n_good


def filter_grid(med, sig, valid):
    """R-D2.  3x3 median over valid cells.  Returns bkg[GY][GX], nse[GY][GX] (+inf where undefined)."""
    GY, GX = med.shape
    bkg = np.zeros((GY, GX)); nse = np.full((GY, GX), np.inf)
    for gy in range(GY):
        for gx in range(GX):
            y0, y1, x0, x1 = max(gy - 1, 0), min(gy + 2, GY), max(gx - 1, 0), min(gx + 2, GX)
            ok = valid[y0:y1, x0:x1]
            if ok.any():
                bkg[gy, gx] = median_rule(med[y0:y1, x0:x1][ok])
                nse[gy, gx] = median_rule(sig[y0:y1, x0:x1][ok])
    return bkg, nse


def _nodes(n_px, G, B):
    """R-D3 along one axis: lower node g0 and fraction t for pixel coordinates 0 .. n_px-1."""
    u = np.clip((np.arange(n_px, dtype=np.float64) - (B - 1) / 2.0) / B, 0.0, G - 1.0)
    g0 = np.minimum(np.floor(u).astype(np.int64), max(G - 2, 0))
    t = u - g0
    g1 = np.minimum(g0 + 1, G - 1)
    return g0, g1, t


def interp_grid(grid, W, H, B=64):
    """R-D3.  Bilinear interpolation of grid[GY][GX] to every pixel; returns (map[H][W], undefined[H][W]) where
    undefined marks pixels with a non-finite interpolation node (their map value is +inf)."""
    grid = np.asarray(grid, dtype=np.float64)
    GY, GX = grid.shape
    x0, x1, tx = _nodes(W, GX, B)
    y0, y1, ty = _nodes(H, GY, B)
    bad = ~np.isfinite(grid)
    g = np.where(bad, 0.0, grid)
    tx = tx[None, :]; ty = ty[:, None]
    top = (1.0 - tx) * g[y0][:, x0] + tx * g[y0][:, x1]
    bot = (1.0 - tx) * g[y1][:, x0] + tx * g[y1][:, x1]
    out = (1.0 - ty) * top + ty * bot
    und = bad[y0][:, x0] | bad[y0][:, x1] | bad[y1][:, x0] | bad[y1][:, x1]
    out[und] = np.inf
    return out, und


def background(cal, mask, B=64, n_min=16):
    """R-D1 + R-D2: the median-filtered background map and its noise map on the cell grid."""
    med, sig, valid, _ = cell_stats(cal, mask, B, n_min)
    return filter_grid(med, sig, valid)


_NEIGH = [(-1, -1), (-1, 0), (-1, 1), (0, -1), (0, 1), (1, -1), (1, 0), (1, 1)]   # (dy, dx), raster order


def detect(cal, mask, bkg, nse, B=64, k_sigma=5.0, slack=0.0):
    """R-D4 .. R-D6.  Returns a dict of arrays over the sources in ascending raster order: x, y, peak, flux, cx, cy,
    bkg, nse, plus the decision margins m_thr = s - max(k * nse, 0) and m_max = min over neighbours of (s_p - s_q)
    (+inf without neighbours).  slack > 0 also returns the near misses (m_thr > -slack and m_max > -slack, ties
    included); the strict set is m_thr > 0 and `strict`."""
    cal = np.asarray(cal, dtype=np.float64)
    good = np.asarray(mask) != 0
    H, W = cal.shape
    bmap, _ = interp_grid(bkg, W, H, B)
    nmap, und = interp_grid(nse, W, H, B)
    s = cal - bmap
    sp = np.full((H + 2, W + 2), -np.inf)              # masked and out-of-frame pixels never win, never count
    sp[1:-1, 1:-1] = np.where(good, s, -np.inf)
    thr = np.maximum(k_sigma * nmap, 0.0)
    m_thr = np.where(good & ~und, s - thr, -np.inf)
    m_max = np.full((H, W), np.inf)
    strict = np.ones((H, W), dtype=bool)
    for i, (dy, dx) in enumerate(_NEIGH):
        q = sp[1 + dy:1 + dy + H, 1 + dx:1 + dx + W]
        with np.errstate(invalid="ignore"):
            d = np.where(np.isfinite(q), s - q, np.inf)
        m_max = np.minimum(m_max, d)
        strict &= (d > 0) if i < 4 else (d >= 0)
    cand = (m_thr > -slack) & (m_max > -slack) if slack > 0 else (m_thr > 0) & strict
    ys, xs = np.nonzero(cand)                          # row-major scan: ascending y * W + x
    flux = np.zeros(xs.size); mx = np.zeros(xs.size); my = np.zeros(xs.size)
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            q = sp[1 + ys + dy, 1 + xs + dx]
            q = np.where(np.isfinite(q), q, 0.0)
            flux += q; mx += q * dx; my += q * dy
    pos = flux > 0
    safe = np.where(pos, flux, 1.0)
    return {"x": xs.astype(np.int32), "y": ys.astype(np.int32), "peak": s[ys, xs], "flux": flux,
            "cx": np.where(pos, mx / safe, 0.0), "cy": np.where(pos, my / safe, 0.0),
            "bkg": bmap[ys, xs], "nse": nmap[ys, xs], "m_thr": m_thr[ys, xs], "m_max": m_max[ys, xs],
            "strict": (m_thr[ys, xs] > 0) & strict[ys, xs]}
