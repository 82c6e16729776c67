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
