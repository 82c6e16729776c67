"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration bench.py times:
configs[1] (all outputs), configs[2] (three frames: lowest dec, belt/cap transition, highest dec; Lanczos-3 +
SIP), configs[3] (coadd of the first three frames) and configs[4] (one frame, nside 2^18, sampled outputs)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import synth  # noqa: E402


@pytest.fixture(scope="module")
def argus():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2207_14304_b200 as a
    a.load_library()
    return a


@pytest.fixture(scope="module")
def ctx(argus):
    c = argus.Context(0)
    c.set_plan_cache(False)
    yield c
    c.close()


def _full_frame_parity(argus, ctx, fr, what, sample=None):
    from gpu_util import assert_values_match, upload
    H, W = fr.shape
    idx_or, dmin = oracle.footprint(fr.wcs, W, H, fr.nside)
    assert dmin > 1e-9, what + ": seeded frame sits on a decision boundary"
    n, idx = argus.argus_healpix_footprint(ctx, fr.wcs, W, H, fr.nside)
    assert n == len(idx_or), what
    assert torch.equal(idx.cpu(), torch.from_numpy(idx_or)), what + ": footprint list differs"
    del idx
    d = upload(fr)
    v = torch.empty(n, dtype=torch.float32, device="cuda")
    w = torch.empty_like(v)
    argus.argus_resample(ctx, fr.wcs, W, H, fr.nside, fr.kernel, v, w, **d)
    torch.cuda.synchronize()
    info = argus.argus_plan_info(ctx)
    vg, wg = v.cpu().numpy(), w.cpu().numpy()
    cal, mask = oracle.calibrate_frame(fr)
    if sample is not None and sample < n:
        rng = np.random.default_rng(0)
        sel = np.sort(rng.choice(n, sample, replace=False))
        idx_or, vg, wg = idx_or[sel], vg[sel], wg[sel]
    vo, wo, fl = oracle.resample(cal, mask, fr.wcs, fr.nside, idx_or, oracle.KERNELS[fr.kernel])
    worst = assert_values_match(vg, wg, vo, wo, fl, what)
    print("%s: n_fp=%d worst=%.3f x tol plan=%s" % (what, n, worst, info))
    return info


def test_config1_full_frame(argus, ctx):
    info = _full_frame_parity(argus, ctx, synth.config1(), "config1")
    assert info["n_footprint"] == 44887802          # SURVEY.md 8(a), confirmed by the oracle
    assert info["n_inside"] > 0.9 * (info["n_tiles"] - info["n_empty"])


def test_config1_full_frame_unit_kernel(argus, ctx):
    """configs[1] through the image-aligned unit kernel (bench.py --unit-kernel), every output against the oracle."""
    ctx.set_fast_path(3)
    try:
        info = _full_frame_parity(argus, ctx, synth.config1(), "config1, unit kernel")
    finally:
        ctx.set_fast_path(1)
    assert info["n_units"] > 20000 and info["n_stray"] == 0


@pytest.mark.parametrize("k", [0, 25, 37])
def test_config2_frames(argus, ctx, k):
    info = _full_frame_parity(argus, ctx, synth.config2_frame(k), "config2[%d]" % k)
    if k == 25:
        assert info["n_exact"] > 0  # the belt/cap ring crosses this frame


def test_config4_one_frame_nside_2p18(argus, ctx):
    _full_frame_parity(argus, ctx, synth.config4_frame(4), "config4[4]", sample=20_000_000)


def test_config3_coadd_full(argus, ctx):
    from gpu_util import assert_coadd_matches, coadd_oracle
    W, H, nside = synth.frames.FULL_W, synth.frames.FULL_H, 1 << 17
    base = synth.config3_frame(0)
    masters = (base.bias, base.dark, base.flat)
    frames = [base] + [synth.config3_frame(k, masters=masters) for k in (1, 2)]
    fps = [oracle.footprint(f.wcs, W, H, nside)[0] for f in frames]
    tiles = np.unique(np.concatenate([fp >> 18 for fp in fps]))
    ppt = 1 << 18
    ref = coadd_oracle(frames, fps, tiles, ppt, nside, "bilinear")
    assert ref["skipped"] == 0
    dt = torch.from_numpy(tiles).cuda()
    s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
    ws = torch.zeros_like(s)
    sk = torch.zeros(1, dtype=torch.int64, device="cuda")
    dm = [torch.from_numpy(m).cuda() for m in masters]
    for f in frames:
        d = dict(raw=torch.from_numpy(f.raw).cuda(), bias=dm[0], dark=dm[1], flat=dm[2], bpm=None, t_exp=f.t_exp,
                 sat_adu=f.sat_adu, flat_min=f.flat_min)
        argus.argus_resample_coadd(ctx, f.wcs, W, H, nside, "bilinear", dt, 256, s, ws, sk, **d)
    torch.cuda.synchronize()
    assert int(sk.item()) == 0
    # every slot except those the oracle flags margin-ambiguous in some frame (R18), to the per-slot R20 tolerance
    worst, n_amb = assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "config3 coadd of 3 frames")
    print("config3 coadd: worst %.3f x tol, %d ambiguous slots of %d pixels accumulated" % (worst, n_amb, ref["n_px"]))


def test_subtract_full_size(argus, ctx):
    """SURVEY 8(f).3 at the size bench.py --workload subtract times (all NSIDE-256 tiles of a configs[3] field, 2^18 pixels
    each, affine match, 5 sigma): the GPU runs the whole layout; the oracle checks 5 of the tiles, every pixel and
    every candidate of them."""
    from test_gpu_subtract import compare
    W, H, nside = synth.frames.FULL_W, synth.frames.FULL_H, 1 << 17
    base = synth.config3_frame(0)
    masters = (base.bias, base.dark, base.flat)
    frames = [base] + [synth.config3_frame(k, masters=masters) for k in (1, 2)]
    wcs = base.wcs
    dm = [torch.from_numpy(m).cuda() for m in masters]
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    tiles = torch.unique(idx >> 18)
    del idx
    ppt = 1 << 18
    pairs = [torch.zeros(tiles.numel() * ppt, dtype=torch.float32, device="cuda") for _ in range(4)]
    for k, f in enumerate(frames):
        d = dict(raw=torch.from_numpy(f.raw).cuda(), bias=dm[0], dark=dm[1], flat=dm[2], bpm=None, t_exp=f.t_exp, sat_adu=f.sat_adu, flat_min=f.flat_min)
        reps = 4 if k < 2 else 1                      # reference: frames 0 and 1, four times each; science: frame 2
        for _ in range(reps):
            argus.argus_resample_coadd(ctx, wcs, W, H, nside, "bilinear", tiles, 256, pairs[2 if k < 2 else 0], pairs[3 if k < 2 else 1], None, **d)
    diff = torch.empty_like(pairs[0]); sig = torch.empty_like(pairs[0])
    nt = tiles.numel()
    al = torch.empty(nt, dtype=torch.float32, device="cuda"); be = torch.empty_like(al)
    nv = torch.empty(nt, dtype=torch.int32, device="cuda")
    cat = torch.zeros((1 << 18) * 32, dtype=torch.uint8, device="cuda")
    kw = dict(match="affine", k_sigma=5.0, read_noise=1.7, gain=1.0, ref_wmin=2.0)
    k = argus.argus_subtract_tiles(ctx, tiles, 256, nside, pairs[0], pairs[1], pairs[2], pairs[3], diff, sig, cat, alpha_out=al,
                                   beta_out=be, nvalid_out=nv, **kw)
    rec = cat.cpu().numpy()[:k * 32].view(argus.TRANSIENT_DTYPE)
    assert np.all(np.diff(rec["pixel"]) > 0)
    th = tiles.cpu().numpy()
    sel = np.unique(np.linspace(0, nt - 1, 5).astype(np.int64))
    cut = lambda t: np.concatenate([t[int(i) * ppt:(int(i) + 1) * ppt].cpu().numpy() for i in sel])
    r = rec[np.isin(rec["tile_rank"], sel)].copy()
    r["tile_rank"] = np.searchsorted(sel, r["tile_rank"])
    g = dict(diff=cut(diff), sig=cut(sig), alpha=al.cpu().numpy()[sel], beta=be.cpu().numpy()[sel], n_valid=nv.cpu().numpy()[sel], rec=r)
    n_must, n_amb = compare(g, th[sel], ppt, nside, [cut(p) for p in pairs], max_ambiguous=10, **kw)
    print("subtract full size: %d tiles, %d candidates; checked tiles %s: %d clear, %d ambiguous" % (nt, k, sel.tolist(), n_must, n_amb))
