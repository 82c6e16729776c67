"""Helpers for the -m gpu parity tests: upload synthetic frames, compare against the oracle."""
import numpy as np
import torch

import oracle
import paper_2207_14304_b200 as argus

VALUE_ATOL, VALUE_RTOL = 1e-3, 1e-5   # BASELINE.json north_star: |d| <= 1e-3 ADU + 1e-5 relative
WEIGHT_ATOL = 1e-5                    # SURVEY.md 8(c)-O6 reading
MAX_AMBIGUOUS_FRAC = 1e-4


def upload(fr, dev="cuda:0"):
    d = dict(raw=torch.from_numpy(fr.raw).to(dev), bias=torch.from_numpy(fr.bias).to(dev),
             dark=torch.from_numpy(fr.dark).to(dev), flat=torch.from_numpy(fr.flat).to(dev),
             bpm=None if fr.bpm is None else torch.from_numpy(fr.bpm).to(dev),
             t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min)
    return d


def gpu_resample_planned(ctx, fr, dfr, kernel=None, w_min=0.5, n_cap=None):
    H, W = fr.shape
    kernel = kernel or fr.kernel
    n, _ = argus.argus_healpix_footprint(ctx, fr.wcs, W, H, fr.nside, want_indices=False)
    cap = n if n_cap is None else n_cap
    v = torch.full((cap,), float("nan"), dtype=torch.float32, device="cuda:0")
    w = torch.full((cap,), float("nan"), dtype=torch.float32, device="cuda:0")
    argus.argus_resample(ctx, fr.wcs, W, H, fr.nside, kernel, v, w, w_min=w_min, **dfr)
    torch.cuda.synchronize()
    return n, v.cpu().numpy(), w.cpu().numpy()


def assert_values_match(v_gpu, w_gpu, v_or, w_or, flag, what="", min_amb_count=0):
    assert np.all(np.isfinite(v_gpu)) and np.all(np.isfinite(w_gpu)), what + ": non-finite output"
    ok = flag == 0
    amb = 1.0 - ok.mean() if len(ok) else 0.0
    # small frames: a couple of ambiguous pixels beside injected defects are more than 1e-4 of a 1e4-pixel footprint
    assert amb <= max(MAX_AMBIGUOUS_FRAC, min_amb_count / max(len(ok), 1)), "%s: %.2e of pixels margin-ambiguous" % (what, amb)
    dv = np.abs(v_gpu[ok] - v_or[ok])
    tol = VALUE_ATOL + VALUE_RTOL * np.abs(v_or[ok])
    worst = (dv / tol).max() if len(dv) else 0.0
    assert worst <= 1.0, "%s: value error %.3f x tolerance (max |d| = %.3e)" % (what, worst, dv.max())
    dw = np.abs(w_gpu[ok] - w_or[ok]).max() if ok.any() else 0.0
    assert dw <= WEIGHT_ATOL, "%s: weight error %.3e" % (what, dw)
    return worst


def oracle_reference(fr, idx, kernel=None, w_min=0.5):
    cal, mask = oracle.calibrate_frame(fr)
    return oracle.resample(cal, mask, fr.wcs, fr.nside, idx, oracle.KERNELS[kernel or fr.kernel], w_min)


def coadd_oracle(frames, fps, tiles, ppt, nside, kernel, w_min=0.5):
    """O7 with the oracle, frame by frame in order, plus what the comparison needs per coadd slot: the tolerance
    (R20) and the "margin-ambiguous in any frame" mask built from the oracle's own per-frame flags (R18).
    Returns dict(sum, wsum, tol_sum, tol_wsum, amb, skipped, n_px)."""
    n_slots = len(tiles) * ppt
    out = dict(sum=np.zeros(n_slots), wsum=np.zeros(n_slots), tol_sum=np.zeros(n_slots), tol_wsum=np.zeros(n_slots),
               amb=np.zeros(n_slots, dtype=bool), skipped=0, n_px=0)
    kern = oracle.KERNELS[kernel]
    for f, fp in zip(frames, fps):
        cal, mask = oracle.calibrate_frame(f)
        v, w, fl = oracle.resample(cal, mask, f.wcs, nside, fp, kern, w_min)
        out["skipped"] += oracle.coadd_accumulate(tiles, ppt, out["sum"], out["wsum"], fp, v, w)
        key = fp // ppt
        rank = np.minimum(np.searchsorted(tiles, key), len(tiles) - 1)
        present = tiles[rank] == key
        slot = (rank * ppt + fp % ppt)[present]          # footprint pixels are unique within a frame
        vp, wp, flp = np.abs(v[present]), w[present], fl[present]
        # R20: |d(w v)| <= w |dv| + |v| |dw|, |dv| <= 1e-3 + 1e-5 |v| (north_star), |dw| <= 1e-5 (R19) and only where
        # w < 1 (w == 1 is exact on both sides, R15); + float32 accumulation, 2^-23 relative per frame
        out["tol_sum"][slot] += wp * (VALUE_ATOL + VALUE_RTOL * vp) + np.where(wp < 1.0, WEIGHT_ATOL * vp, 0.0) + 2.0 ** -23 * wp * vp
        out["tol_wsum"][slot] += np.where((wp < 1.0) & (wp > 0.0), WEIGHT_ATOL, 0.0) + 2.0 ** -23 * wp
        out["amb"][slot[flp != 0]] = True
        out["n_px"] += int(present.sum())
    return out


def assert_coadd_matches(s_gpu, w_gpu, ref, what="", min_amb_count=8):
    """Every slot that is not margin-ambiguous in some frame (the oracle's flags, R18) must meet R20; the flagged
    slots are counted and bounded like the single-frame rule (< 1e-4 of the pixels accumulated)."""
    sg, wg = s_gpu.astype(np.float64), w_gpu.astype(np.float64)
    assert np.all(np.isfinite(sg)) and np.all(np.isfinite(wg)), what + ": non-finite coadd"
    ok = ~ref["amb"]
    n_amb = int(ref["amb"].sum())
    assert n_amb <= max(MAX_AMBIGUOUS_FRAC * ref["n_px"], min_amb_count), "%s: %d slots margin-ambiguous" % (what, n_amb)
    dw = np.abs(wg - ref["wsum"])[ok]
    assert np.all(dw <= ref["tol_wsum"][ok] + 1e-12), "%s: wsum error %.3e" % (what, dw.max())
    ds = np.abs(sg - ref["sum"])[ok]
    tol = ref["tol_sum"][ok]
    bad = ds > tol + 1e-12
    worst = (ds[tol > 0] / tol[tol > 0]).max() if (tol > 0).any() else 0.0
    assert not bad.any(), "%s: %d slots outside the coadd tolerance, worst %.3f x (max |d| = %.3e)" % (what, int(bad.sum()), worst, ds.max())
    return worst, n_amb
