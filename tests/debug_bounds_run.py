"""Run under ARGUS_LIBRARY=libargus_debug.so (the ARGUS_DEBUG_BOUNDS build) by tests/test_gpu_debug_bounds.py: every
planned path with staged source boxes -- tile kernel (bilinear, Lanczos-3, coadd), unit kernel (raw and pre-fused masters,
coadd, forced strays) -- on config 0, the special pointings and 8 fuzz geometries.  Every shared-memory gather index is
checked on the device against its staged box; a violation is latched and makes argus_plan_info fail.  Not a test file
itself (no oracle comparison here: the parity tests do that with the product build)."""
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import paper_2207_14304_b200 as argus  # noqa: E402
import synth  # noqa: E402
from gpu_util import upload  # noqa: E402


def main():
    assert os.environ.get("ARGUS_LIBRARY", "").endswith("libargus_debug.so")
    ctx = argus.Context(0)
    n_runs = 0

    def run(fr, kernels=("bilinear", "lanczos3"), modes=(1, 2, 3)):
        nonlocal n_runs
        H, W = fr.shape
        d = upload(fr)
        n, idx = argus.argus_healpix_footprint(ctx, fr.wcs, W, H, fr.nside)
        v = torch.empty(max(n, 1), dtype=torch.float32, device="cuda")
        w = torch.empty_like(v)
        tiles = torch.unique(idx >> 18) if fr.nside >= (1 << 14) and n else None
        for mode in modes:
            ctx.set_fast_path(mode)
            for k in kernels:
                argus.argus_resample(ctx, fr.wcs, W, H, fr.nside, k, v, w, **d)
                if tiles is not None:
                    ppt = (fr.nside // (fr.nside >> 9)) ** 2
                    s = torch.zeros(tiles.numel() * ppt, dtype=torch.float32, device="cuda")
                    argus.argus_resample_coadd(ctx, fr.wcs, W, H, fr.nside, k, tiles >> 0, fr.nside >> 9, s, torch.zeros_like(s), None, **d)
                n_runs += 1
            if fr.bpm is None:
                off, gain = argus.argus_prepare_masters(ctx, d["bias"], d["dark"], d["flat"], None, fr.t_exp, fr.flat_min)
                argus.argus_resample(ctx, fr.wcs, W, H, fr.nside, "bilinear", v, w, raw=d["raw"], offset=off, gain=gain, sat_adu=fr.sat_adu)
        ctx.set_fast_path(1)
        torch.cuda.synchronize()
        argus.argus_plan_info(ctx)         # raises if any gather left its box (or anything overflowed)

    cfg0 = synth.config0()
    if "--expect-violation" in sys.argv:   # self-test of the check: it must fire when the box is pretended 24 cells narrower
        ctx.set_unit_margin(32)
        try:
            run(cfg0, kernels=("bilinear",), modes=(3,))
        except argus.ArgusError as e:
            print("violation detected: %s" % e)
            return
        raise SystemExit("the bounds check did not fire")
    run(cfg0)
    run(synth.inject_defects(cfg0))
    ctx.set_unit_margin(-2)                # forced strays
    run(cfg0, kernels=("bilinear",), modes=(3,))
    ctx.set_unit_margin(0)
    for name, (crval, rot, nside) in synth.special_pointings().items():
        run(synth.make_frame(7, 512, 512, 100, synth.make_wcs(crval, (255.5, 255.5), rot), nside, "bilinear"))
    for seed in range(8):
        rng = np.random.default_rng(1000 + seed)
        nside = 1 << int(rng.integers(14, 19))
        hp = math.degrees(math.sqrt(4 * math.pi / (12.0 * nside * nside)))
        W, H = int(rng.integers(12, 48)) * 8, int(rng.integers(90, 380))
        dec = math.degrees(math.asin(rng.uniform(-1, 1)))
        wcs = synth.make_wcs((rng.uniform(0, 360), dec), ((W - 1) / 2.0, (H - 1) / 2.0), rng.uniform(-180, 180), scale_deg=hp / rng.uniform(0.6, 2.5))
        run(synth.make_frame(2000 + seed, W, H, 60, wcs, nside, "bilinear"))
    ctx.close()
    print("debug bounds ok: %d frame x kernel x path runs, no gather outside its staged box" % n_runs)


if __name__ == "__main__":
    main()
