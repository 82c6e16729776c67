"""GPU parity (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle, element by
element on the same seeded inputs.  Footprints bit-exact; values within 1e-3 ADU + 1e-5 relative."""
import math

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
    yield c
    c.close()


def test_calibrate_matches_oracle(argus, ctx):
    from gpu_util import upload
    fr = synth.inject_defects(synth.config0())
    d = upload(fr)
    cal, mask = argus.argus_calibrate(ctx, d["raw"], d["bias"], d["dark"], d["flat"], d["bpm"], fr.t_exp, fr.sat_adu, fr.flat_min)
    torch.cuda.synchronize()
    oc, om = oracle.calibrate_frame(fr)
    assert np.array_equal(mask.cpu().numpy(), om)
    dv = np.abs(cal.cpu().numpy().astype(np.float64) - oc)
    assert np.all(dv <= 1e-3 + 1e-5 * np.abs(oc))
    assert om.sum() < om.size  # the defects are really there
    # odd width: scalar path
    fr2 = synth.make_frame(3, 37, 19, 5, fr.wcs, fr.nside, "bilinear")
    d2 = upload(fr2)
    cal2, mask2 = argus.argus_calibrate(ctx, d2["raw"], d2["bias"], d2["dark"], d2["flat"], None, fr2.t_exp)
    oc2, om2 = oracle.calibrate_frame(fr2)
    assert np.array_equal(mask2.cpu().numpy(), om2)
    assert np.all(np.abs(cal2.cpu().numpy() - oc2) <= 1e-3 + 1e-5 * np.abs(oc2))


def test_config0_footprint_bit_exact(argus, ctx, cfg0, cfg0_fp):
    idx_or, dmin = cfg0_fp
    n, idx = argus.argus_healpix_footprint(ctx, cfg0.wcs, 512, 512, cfg0.nside)
    assert n == len(idx_or)
    assert np.array_equal(idx.cpu().numpy(), idx_or)
    info = argus.argus_plan_info(ctx)
    assert info["n_footprint"] == n and info["n_inside"] > 0 and info["n_border"] > 0


@pytest.mark.parametrize("kernel", ["bilinear", "lanczos3"])
def test_config0_values(argus, ctx, cfg0, cfg0_fp, kernel):
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    idx_or, _ = cfg0_fp
    d = upload(cfg0)
    n, v, w = gpu_resample_planned(ctx, cfg0, d, kernel)
    assert n == len(idx_or)
    vo, wo, fl = oracle_reference(cfg0, idx_or, kernel)
    assert_values_match(v, w, vo, wo, fl, "config0 planned " + kernel)
    # general list path (explicit idx, FP64 coordinates), shuffled order
    rng = np.random.default_rng(0)
    perm = rng.permutation(len(idx_or))[:50000]
    sub = torch.from_numpy(idx_or[perm]).cuda()
    v2 = torch.empty(len(perm), dtype=torch.float32, device="cuda")
    w2 = torch.empty_like(v2)
    argus.argus_resample(ctx, cfg0.wcs, 512, 512, cfg0.nside, kernel, v2, w2, idx=sub, **d)
    torch.cuda.synchronize()
    assert_values_match(v2.cpu().numpy(), w2.cpu().numpy(), vo[perm], wo[perm], fl[perm], "config0 list " + kernel)


def test_p10_fused_equals_unfused(argus, ctx, cfg0, cfg0_fp):
    from gpu_util import gpu_resample_planned, upload
    d = upload(cfg0)
    n, v, w = gpu_resample_planned(ctx, cfg0, d, "bilinear")
    cal, mask = argus.argus_calibrate(ctx, d["raw"], d["bias"], d["dark"], d["flat"], None, cfg0.t_exp)
    n2, v2, w2 = gpu_resample_planned(ctx, cfg0, dict(cal=cal, mask=mask), "bilinear")
    assert n == n2
    # the fused call runs the TMA-staged kernel, the unfused one the general kernel: their tile-local coordinate
    # arithmetic differs by ~2e-7 px, hence "1 ulp-level" rather than bit equality
    assert np.all(np.abs(w - w2) <= 2e-6)
    assert np.array_equal(w == 1.0, w2 == 1.0) and np.array_equal(w == 0.0, w2 == 0.0)
    assert np.all(np.abs(v - v2) <= 1e-4 + 2e-6 * np.abs(v))
    # same kernel on both sides (fast path off): calibration fused or not must agree to rounding
    ctx.set_fast_path(False)
    try:
        n3, v3, w3 = gpu_resample_planned(ctx, cfg0, d, "bilinear")
    finally:
        ctx.set_fast_path(True)
    assert np.array_equal(w3, w2)
    assert np.all(np.abs(v3 - v2) <= 1e-6 * np.maximum(1.0, np.abs(v3)))


def test_mask_logic_frame(argus, ctx):
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    fr = synth.inject_defects(synth.config0())
    idx_or, _ = oracle.footprint(fr.wcs, 512, 512, fr.nside)
    d = upload(fr)
    for kernel, w_min in (("bilinear", 0.5), ("bilinear", 1.0), ("lanczos3", 0.5)):
        n, v, w = gpu_resample_planned(ctx, fr, d, kernel, w_min)
        vo, wo, fl = oracle_reference(fr, idx_or, kernel, w_min)
        assert (wo < 1).sum() > 100 and (wo == 0).sum() > 10
        assert_values_match(v, w, vo, wo, fl, "defects %s w_min=%g" % (kernel, w_min))


@pytest.mark.parametrize("name", sorted(synth.special_pointings()))
def test_special_pointings(argus, ctx, name):
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    crval, rot, nside = synth.special_pointings()[name]
    W = H = 512
    wcs = synth.make_wcs(crval, (255.5, 255.5), rot)
    fr = synth.make_frame(77, W, H, 200, wcs, nside, "bilinear")
    idx_or, dmin = oracle.footprint(wcs, W, H, nside)
    assert dmin > 1e-9, "seeded pointing sits on a decision boundary; re-seed"
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    assert n == len(idx_or), name
    assert np.array_equal(idx.cpu().numpy(), idx_or), name
    d = upload(fr)
    n, v, w = gpu_resample_planned(ctx, fr, d, "bilinear")
    vo, wo, fl = oracle_reference(fr, idx_or, "bilinear")
    assert_values_match(v, w, vo, wo, fl, name)


def test_sip_and_rectangular_odd_width(argus, ctx):
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    rng = np.random.default_rng(5)
    W, H = 601, 333  # W % 4 != 0 -> scalar staging path
    sip = synth.make_sip(rng, 3, 300.0)
    sip = (3, sip[1] * 30, sip[2] * 30)
    wcs = synth.make_wcs((211.0, 47.0), ((W - 1) / 2, (H - 1) / 2), 23.0, sip=sip)
    fr = synth.make_frame(9, W, H, 150, wcs, 1 << 17, "bilinear")
    idx_or, dmin = oracle.footprint(wcs, W, H, fr.nside)
    assert dmin > 1e-9
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, fr.nside)
    assert np.array_equal(idx.cpu().numpy(), idx_or)
    d = upload(fr)
    for kernel in ("bilinear", "lanczos3"):
        n, v, w = gpu_resample_planned(ctx, fr, d, kernel)
        vo, wo, fl = oracle_reference(fr, idx_or, kernel)
        assert_values_match(v, w, vo, wo, fl, "sip " + kernel)


def test_small_nside_coarse_wcs(argus, ctx):
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    nside = 1 << 10
    hp = math.degrees(math.sqrt(4 * math.pi / (12.0 * nside * nside)))
    W = H = 256
    wcs = synth.make_wcs((75.0, -33.0), (127.5, 127.5), 12.0, scale_deg=hp / 1.2)
    fr = synth.make_frame(4, W, H, 50, wcs, nside, "bilinear")
    idx_or, dmin = oracle.footprint(wcs, W, H, nside)
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    assert np.array_equal(idx.cpu().numpy(), idx_or)
    d = upload(fr)
    n, v, w = gpu_resample_planned(ctx, fr, d, "bilinear")
    vo, wo, fl = oracle_reference(fr, idx_or, "bilinear")
    assert_values_match(v, w, vo, wo, fl, "nside 2^10")


def test_lanczos_saturated_stars_handover(argus, ctx):
    """Saturated star cores: masked pixels next to ~6e4-ADU taps.  The Lanczos-3 fast kernel hands such tiles to the
    FP64 general kernel at run time (and keeps the others); both kernels, planned path, must meet the tolerance,
    and the fast path must agree with the general kernel alone."""
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    W = H = 512
    fr = _saturated_star_frame()
    wcs = fr.wcs
    idx_or, dmin = oracle.footprint(wcs, W, H, fr.nside)
    d = upload(fr)
    for kernel in ("lanczos3", "bilinear"):
        n, v, w = gpu_resample_planned(ctx, fr, d, kernel)
        vo, wo, fl = oracle_reference(fr, idx_or, kernel)
        assert (wo < 1).sum() > 50
        assert_values_match(v, w, vo, wo, fl, "saturated stars " + kernel)
        ctx.set_fast_path(False)
        try:
            n2, v2, w2 = gpu_resample_planned(ctx, fr, d, kernel)
        finally:
            ctx.set_fast_path(True)
        assert_values_match(v2, w2, vo, wo, fl, "saturated stars, general kernel " + kernel)


def test_plan_overlap_option_and_stream_order(argus, ctx, cfg0, cfg0_fp):
    """Plans built on the side streams (default) and in place must give identical outputs; results follow the
    caller's stream order when frames with different WCS are enqueued back to back without synchronisation."""
    from gpu_util import upload
    d = upload(cfg0)
    wcs2 = synth.make_wcs((30.01, 20.02), (255.5, 255.5), 7.0)
    outs = {}
    for overlap in (True, False):
        ctx.set_plan_overlap(overlap)
        ctx.set_plan_cache(False)
        try:
            res = []
            for k in range(6):   # alternate two pointings, never synchronise in between
                wcs = cfg0.wcs if k % 2 == 0 else wcs2
                v = torch.full((200000,), float("nan"), dtype=torch.float32, device="cuda")
                w = torch.full_like(v, float("nan"))
                argus.argus_resample(ctx, wcs, 512, 512, cfg0.nside, "bilinear", v, w, **d)
                res.append((v, w))
            torch.cuda.synchronize()
            outs[overlap] = [(v.cpu().numpy(), w.cpu().numpy()) for v, w in res]
        finally:
            ctx.set_plan_overlap(True)
            ctx.set_plan_cache(True)
    for k in range(6):
        assert np.array_equal(outs[True][k][0], outs[False][k][0], equal_nan=True)
        assert np.array_equal(outs[True][k][1], outs[False][k][1], equal_nan=True)
    n0 = len(cfg0_fp[0])
    assert np.isfinite(outs[True][0][0][:n0]).all() and np.isnan(outs[True][0][0][n0:]).all()
    assert np.array_equal(outs[True][0][0], outs[True][2][0], equal_nan=True)   # same pointing, same result
    assert not np.array_equal(outs[True][0][0], outs[True][1][0], equal_nan=True)


@pytest.mark.parametrize("seed", range(int(__import__("os").environ.get("ARGUS_FUZZ_SEEDS", "48"))))
def test_random_geometry_fuzz(argus, ctx, seed):
    """Seeded random pointings, rotations, pixel scales, nside, frame shapes, SIP and kernels: footprint bit-exact,
    values within tolerance.  Exercises sheared / oversized tiles (slow list), both fast kernels and the flat plan."""
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    rng = np.random.default_rng(1000 + seed)
    nside = 1 << int(rng.integers(14, 19))
    hp = math.degrees(math.sqrt(4 * math.pi / (12.0 * nside * nside)))
    scale = hp / rng.uniform(0.6, 2.5)            # HEALPix pixel = 0.6 .. 2.5 detector pixels
    W = int(rng.integers(12, 48)) * 8 if rng.random() < 0.7 else int(rng.integers(100, 380))
    H = int(rng.integers(90, 380))
    dec = math.degrees(math.asin(rng.uniform(-1, 1)))
    if seed % 6 == 0:
        dec = math.copysign(89.0 + rng.uniform(0, 0.99), dec)        # polar caps, near the poles
    crval = (rng.uniform(0, 360), dec)
    sip = None
    if rng.random() < 0.5:
        o, ap, bp = synth.make_sip(rng, 3, W / 2.0)
        sip = (o, ap * 20, bp * 20)
    wcs = synth.make_wcs(crval, ((W - 1) / 2.0 + rng.uniform(-0.5, 0.5), (H - 1) / 2.0 + rng.uniform(-0.5, 0.5)),
                         rng.uniform(-180, 180), scale_deg=scale, sip=sip)
    kernel = "lanczos3" if rng.random() < 0.4 else "bilinear"
    fr = synth.make_frame(2000 + seed, W, H, 60, wcs, nside, kernel)
    if seed % 3 == 0:
        fr = synth.inject_defects(fr)
    idx_or, dmin = oracle.footprint(wcs, W, H, nside)
    if dmin <= 1e-9:
        pytest.skip("seeded pointing sits on a decision boundary")
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    assert n == len(idx_or)
    assert np.array_equal(idx.cpu().numpy(), idx_or)
    d = upload(fr)
    n, v, w = gpu_resample_planned(ctx, fr, d, kernel)
    vo, wo, fl = oracle_reference(fr, idx_or, kernel)
    assert_values_match(v, w, vo, wo, fl, "fuzz %d %s nside 2^%d %dx%d dec %.2f" % (seed, kernel, int(math.log2(nside)), W, H, dec),
                        min_amb_count=8)


def test_tiny_nside_flat_plan(argus, ctx):
    """nside < 256 has no 8x8-tile blocks: the flat plan (one fit per tile) must give the same parity."""
    from gpu_util import assert_values_match, gpu_resample_planned, oracle_reference, upload
    nside = 1 << 7
    hp = math.degrees(math.sqrt(4 * math.pi / (12.0 * nside * nside)))
    W = H = 128
    wcs = synth.make_wcs((222.0, 31.0), (63.5, 63.5), -7.0, scale_deg=hp / 1.3)
    fr = synth.make_frame(6, W, H, 30, wcs, nside, "bilinear")
    idx_or, dmin = oracle.footprint(wcs, W, H, nside)
    assert dmin > 1e-9
    n, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    assert np.array_equal(idx.cpu().numpy(), idx_or)
    d = upload(fr)
    n, v, w = gpu_resample_planned(ctx, fr, d, "bilinear")
    vo, wo, fl = oracle_reference(fr, idx_or, "bilinear")
    assert_values_match(v, w, vo, wo, fl, "nside 2^7")


def test_coadd_three_frames(argus, ctx):
    from gpu_util import assert_coadd_matches, coadd_oracle, upload
    W = H = 512
    nside = 1 << 17
    frames = [synth.config3_frame(k, W, H) for k in range(3)]
    fps = [oracle.footprint(f.wcs, W, H, nside)[0] for f in frames]
    tiles = np.unique(np.concatenate([fp >> 18 for fp in fps]))[:-1]  # drop one tile: exercises "skipped"
    ppt = 1 << 18
    ref = coadd_oracle(frames, fps, tiles, ppt, nside, "bilinear")
    dt = torch.from_numpy(tiles).cuda()
    for fused in (True, False):
        s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
        ws = torch.zeros_like(s)
        sk = torch.zeros(1, dtype=torch.int64, device="cuda")
        for f, fp in zip(frames, fps):
            d = upload(f)
            if fused:
                argus.argus_resample_coadd(ctx, f.wcs, W, H, nside, "bilinear", dt, 256, s, ws, sk, **d)
            else:
                n, idx = argus.argus_healpix_footprint(ctx, f.wcs, W, H, nside)
                v = torch.empty(n, dtype=torch.float32, device="cuda")
                w = torch.empty_like(v)
                argus.argus_resample(ctx, f.wcs, W, H, nside, "bilinear", v, w, **d)
                argus.argus_coadd_accumulate(ctx, dt, 256, nside, s, ws, idx, v, w, sk)
        torch.cuda.synchronize()
        assert int(sk.item()) == ref["skipped"] > 0
        assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "coadd of 3 frames, fused=%s" % fused)


@pytest.mark.parametrize("force_unit", [False, True])
def test_coadd_buffers_aligned_to_4_bytes_only(argus, ctx, force_unit):
    """The header asks for float alignment of sum / wsum, nothing more; the kernels' L2 prefetch of the accumulators needs
    16 bytes and must step aside: accumulators that start 4 bytes into an allocation give the bits of aligned ones."""
    from gpu_util import upload
    W = H = 512
    nside = 1 << 17
    f = synth.config3_frame(0, W, H)
    fp = oracle.footprint(f.wcs, W, H, nside)[0]
    tiles = np.unique(fp >> 18)
    ppt = 1 << 18
    dt = torch.from_numpy(tiles).cuda()
    d = upload(f)
    if force_unit:
        ctx.set_fast_path(3)
    try:
        out = []
        for shift in (0, 1):
            s = torch.zeros(len(tiles) * ppt + 4, dtype=torch.float32, device="cuda")
            ws = torch.zeros_like(s)
            sv, wv = s[shift:shift + len(tiles) * ppt], ws[shift:shift + len(tiles) * ppt]
            assert sv.data_ptr() % 16 == 4 * shift
            for _ in range(2):
                argus.argus_resample_coadd(ctx, f.wcs, W, H, nside, "bilinear", dt, 256, sv, wv, None, **d)
            torch.cuda.synchronize()
            out.append((sv.clone(), wv.clone()))
    finally:
        if force_unit:
            ctx.set_fast_path(1)
    assert torch.equal(out[0][0].view(torch.int32), out[1][0].view(torch.int32)) and torch.equal(out[0][1], out[1][1])
    assert float(out[0][1].sum()) > 0


def _saturated_star_frame(seed=11, kernel="lanczos3"):
    """512 x 512 frame with six stars whose cores clip at 65535 (=> masked) and wings up to ~6e4 ADU."""
    W = H = 512
    wcs = synth.make_wcs((30.0, 20.0), (255.5, 255.5), 0.3)
    fr = synth.make_frame(seed, W, H, 40, wcs, 1 << 17, kernel)
    rng = np.random.default_rng(3)
    raw = fr.raw.astype(np.float64)
    yy, xx = np.mgrid[0:H, 0:W]
    for _ in range(6):
        sx, sy = rng.uniform(20, W - 20, 2)
        raw += 4e5 * np.exp(-0.5 * ((xx - sx) ** 2 + (yy - sy) ** 2) / 0.85 ** 2)
    fr.raw = np.clip(np.rint(raw), 0, 65535).astype(np.uint16)
    assert (fr.raw == 65535).sum() > 10
    return fr


def test_coadd_lanczos_fused(argus, ctx):
    """Fused calibrate + Lanczos-3 resample + accumulate (fast kernel, COADD variant) against the oracle."""
    from gpu_util import assert_coadd_matches, coadd_oracle, upload
    W = H = 512
    nside = 1 << 17
    frames = [synth.config3_frame(k, W, H) for k in range(2)]
    fps = [oracle.footprint(f.wcs, W, H, nside)[0] for f in frames]
    tiles = np.unique(np.concatenate([fp >> 18 for fp in fps]))
    ppt = 1 << 18
    ref = coadd_oracle(frames, fps, tiles, ppt, nside, "lanczos3")
    assert ref["skipped"] == 0
    dt = torch.from_numpy(tiles).cuda()
    s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
    ws = torch.zeros_like(s)
    for f in frames:
        argus.argus_resample_coadd(ctx, f.wcs, W, H, nside, "lanczos3", dt, 256, s, ws, None, **upload(f))
    torch.cuda.synchronize()
    assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "Lanczos-3 coadd of 2 dithered frames")


def test_coadd_lanczos_repeated_wcs_cached_plan(argus, ctx):
    """The Lanczos-3 fast kernel hands tiles with masked + bright pixels to the general kernel at run time by appending
    to the plan's slow list.  With an identical WCS the cached plan is reused: the list must be back in the plan's
    state for every call, or the (non-idempotent) coadd accumulation counts those tiles twice."""
    from gpu_util import assert_coadd_matches, coadd_oracle, upload
    W = H = 512
    nside = 1 << 17
    fr = _saturated_star_frame()
    fp = oracle.footprint(fr.wcs, W, H, nside)[0]
    tiles = np.unique(fp >> 18)
    ppt = 1 << 18
    n_calls = 3
    ref = coadd_oracle([fr] * n_calls, [fp] * n_calls, tiles, ppt, nside, "lanczos3")
    dt = torch.from_numpy(tiles).cuda()
    d = upload(fr)
    s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
    ws = torch.zeros_like(s)
    ctx.set_plan_cache(True)
    launches = []
    for _ in range(n_calls):
        l0 = ctx.launch_count()
        argus.argus_resample_coadd(ctx, fr.wcs, W, H, nside, "lanczos3", dt, 256, s, ws, None, **d)
        launches.append(ctx.launch_count() - l0)
    torch.cuda.synchronize()
    assert launches[1] == launches[2] < launches[0], "calls 2 and 3 must reuse the cached plan: %r" % (launches,)
    argus.argus_plan_info(ctx)     # no overflow (the slow list did not grow from call to call)
    assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "Lanczos-3 coadd, same WCS three times")
    # value + weight form through the same cached plan: identical results call after call
    n = len(fp)
    outs = []
    for _ in range(3):
        v = torch.full((n,), float("nan"), dtype=torch.float32, device="cuda")
        w = torch.full_like(v, float("nan"))
        argus.argus_resample(ctx, fr.wcs, W, H, nside, "lanczos3", v, w, **d)
        outs.append((v.cpu().numpy(), w.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[2][0]) and np.array_equal(outs[0][1], outs[2][1])


def test_lanczos_fine_grid_two_stage_form(argus, ctx):
    """nside 2^18 at the configs' pixel scale: every tile's source box fits 48 x 48 pixels, so the tile kernel runs its
    two-stage Lanczos-3 form (FastCfg<1, 1>, resample_fast.cuh).  Values + weights and a coadd of three calls against
    the oracle, on a frame with saturated stars (run-time hand-over to the FP64 kernel); values + weights bit for bit
    against the one-stage form (ARGUS_OPT_FAST_PATH = 4): the same arithmetic per tile in another pipeline."""
    from gpu_util import (assert_coadd_matches, assert_values_match, coadd_oracle, gpu_resample_planned,
                          oracle_reference, upload)
    W = H = 512
    fr = _saturated_star_frame()
    fr.nside = nside = 1 << 18
    fp, _ = oracle.footprint(fr.wcs, W, H, nside)
    d = upload(fr)
    n, v, w = gpu_resample_planned(ctx, fr, d, "lanczos3")
    assert n == len(fp)
    vo, wo, fl = oracle_reference(fr, fp, "lanczos3")
    assert (wo < 1).sum() > 100
    assert_values_match(v, w, vo, wo, fl, "nside 2^18 Lanczos-3, two-stage form")
    ppt = (nside // 256) ** 2                 # pixels of an NSIDE-256 coadd tile: 2^20 at nside 2^18
    tiles = np.unique(fp // ppt)
    ref = coadd_oracle([fr] * 3, [fp] * 3, tiles, ppt, nside, "lanczos3")
    dt = torch.from_numpy(tiles).cuda()

    def coadd():
        s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
        ws = torch.zeros_like(s)
        for _ in range(3):
            argus.argus_resample_coadd(ctx, fr.wcs, W, H, nside, "lanczos3", dt, 256, s, ws, None, **d)
        torch.cuda.synchronize()
        return s.cpu().numpy(), ws.cpu().numpy()

    s2, w2 = coadd()
    assert_coadd_matches(s2, w2, ref, "nside 2^18 Lanczos-3 coadd, two-stage form")
    ctx.set_fast_path(4)
    try:
        n1, v1, w1 = gpu_resample_planned(ctx, fr, d, "lanczos3")
        s1, ws1 = coadd()
    finally:
        ctx.set_fast_path(True)
    assert n1 == n and np.array_equal(v1, v) and np.array_equal(w1, w)
    # the coadd instantiations of the two forms are compiled apart and differ by single roundings (1 ulp on some 4e-3 of the
    # slots): each is held to the oracle, and the same tiles must have been handed over (weights equal to rounding)
    assert_coadd_matches(s1, ws1, ref, "nside 2^18 Lanczos-3 coadd, one-stage form")
    assert np.abs(ws1 - w2).max() <= 3 * 2.0 ** -22 and np.abs(s1 - s2).max() <= 3 * 2.0 ** -13


def test_overflow_of_an_earlier_frame_is_latched(argus, cfg0):
    """An output-capacity overflow of frame k must still be reported when the check comes after frame k + 1 was planned
    (plan statistics live in rotating scratch sets; the error is latched context-wide until read)."""
    from gpu_util import upload
    c = argus.Context(0)
    try:
        d = upload(cfg0)
        wcs2 = synth.make_wcs((30.01, 20.02), (255.5, 255.5), 7.0)
        small = torch.zeros(1000, dtype=torch.float32, device="cuda")
        small_w = torch.zeros_like(small)
        big = torch.zeros(400000, dtype=torch.float32, device="cuda")
        big_w = torch.zeros_like(big)
        for overlap in (True, False):
            c.set_plan_overlap(overlap)
            argus.argus_resample(c, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", small, small_w, **d)   # overflows
            argus.argus_resample(c, wcs2, 512, 512, cfg0.nside, "bilinear", big, big_w, **d)             # fits
            with pytest.raises(argus.ArgusError) as e:
                argus.argus_plan_info(c)
            assert e.value.status == -6
            info = argus.argus_plan_info(c)       # reading cleared the latch; the second frame's plan is intact
            assert 0 < info["n_footprint"] <= 400000
    finally:
        c.close()


def test_resample_host_matches_device_path(argus, ctx, cfg0, cfg0_fp):
    """C-ABI entry with HOST buffers: same outputs as the device-buffer call, over several pipelined frames."""
    from gpu_util import upload
    d = upload(cfg0)
    n = len(cfg0_fp[0])
    v = torch.empty(n, dtype=torch.float32, device="cuda")
    w = torch.empty_like(v)
    argus.argus_resample(ctx, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", v, w, **d)
    torch.cuda.synchronize()
    h_raw = torch.from_numpy(cfg0.raw).pin_memory()
    outs = [(torch.full((n,), float("nan")).pin_memory(), torch.full((n,), float("nan")).pin_memory()) for _ in range(5)]
    for hv, hw in outs:
        argus.argus_resample_host(ctx, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", n, h_raw, hv, hw, bias=d["bias"],
                                  dark=d["dark"], flat=d["flat"], t_exp=cfg0.t_exp, sat_adu=cfg0.sat_adu, flat_min=cfg0.flat_min)
    argus.argus_host_wait(ctx)
    for hv, hw in outs:
        assert torch.equal(hv, v.cpu()) and torch.equal(hw, w.cpu())


def test_plan_scratch_overflow_is_reported(argus):
    """A context too small for the frame's tiles reports ARGUS_ERR_CAPACITY instead of writing out of bounds."""
    small = argus.Context(0, max_tiles=64)
    try:
        fr = synth.config0()
        with pytest.raises(argus.ArgusError) as e:
            argus.argus_healpix_footprint(small, fr.wcs, 512, 512, fr.nside)
        assert e.value.status == -6
    finally:
        small.close()


def test_capacity_and_errors(argus, ctx, cfg0):
    from gpu_util import upload
    d = upload(cfg0)
    v = torch.zeros(1000, dtype=torch.float32, device="cuda")
    w = torch.zeros_like(v)
    argus.argus_resample(ctx, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", v, w, **d)  # footprint >> 1000
    with pytest.raises(argus.ArgusError) as e:
        argus.argus_plan_info(ctx)
    assert e.value.status == -6
    with pytest.raises(argus.ArgusError):
        argus.argus_healpix_footprint(ctx, cfg0.wcs, 512, 512, 1000)  # nside not a power of two
    bad = synth.make_wcs((0, 0), (0, 0), 0.0, scale_deg=0.0)
    with pytest.raises(argus.ArgusError):
        argus.argus_healpix_footprint(ctx, bad, 512, 512, 1 << 17)
    # frame that does not see the sky region at all is impossible (every TAN frame has a footprint), but a
    # 1x1 frame must work: footprint of 0 or 1 pixels
    n, idx = argus.argus_healpix_footprint(ctx, synth.make_wcs((10, 10), (0, 0), 0.0), 1, 1, 1 << 17)
    n_or = len(oracle.footprint(synth.make_wcs((10, 10), (0, 0), 0.0), 1, 1, 1 << 17)[0])
    assert n == n_or


@pytest.mark.parametrize("defects", [False, True])
def test_unit_kernel_forced(argus, cfg0, cfg0_fp, defects):
    """The image-aligned unit kernel (resample_unit.cuh) on config 0, where the default choice is the tile kernel:
    ARGUS_OPT_FAST_PATH = 3.  Value + weight form and the fused coadd form, clean and with defects (saturated block, low /
    NaN flat: the masked loop; a bad-pixel mask sends the frame to the general kernel, so the bpm is dropped here)."""
    from gpu_util import assert_coadd_matches, assert_values_match, coadd_oracle, gpu_resample_planned, oracle_reference, upload
    c = argus.Context(0)
    try:
        c.set_fast_path(3)
        fr = cfg0
        if defects:
            fr = synth.inject_defects(cfg0)
            fr.bpm = None
        idx_or = cfg0_fp[0]
        d = upload(fr)
        n, v, w = gpu_resample_planned(c, fr, d, "bilinear")
        info = argus.argus_plan_info(c)
        assert info["n_units"] > 0 and info["n_stray"] == 0
        vo, wo, fl = oracle_reference(fr, idx_or, "bilinear")
        assert_values_match(v, w, vo, wo, fl, "unit kernel, config 0, defects=%s" % defects, min_amb_count=8)
        n, v, w = gpu_resample_planned(c, fr, d, "lanczos3")
        assert argus.argus_plan_info(c)["n_units"] > 0
        vo, wo, fl = oracle_reference(fr, idx_or, "lanczos3")
        assert_values_match(v, w, vo, wo, fl, "unit kernel, Lanczos-3, config 0, defects=%s" % defects, min_amb_count=8)
        tiles = np.unique(idx_or >> 18)[1:]            # one tile absent from the layout
        ppt = 1 << 18
        ref = coadd_oracle([fr, fr], [idx_or, idx_or], tiles, ppt, fr.nside, "bilinear")
        s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
        ws = torch.zeros_like(s)
        sk = torch.zeros(1, dtype=torch.int64, device="cuda")
        for _ in range(2):
            argus.argus_resample_coadd(c, fr.wcs, 512, 512, fr.nside, "bilinear", torch.from_numpy(tiles).cuda(), 256, s, ws, sk, **d)
        torch.cuda.synchronize()
        assert int(sk.item()) == ref["skipped"] > 0
        assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "unit kernel coadd, defects=%s" % defects)
    finally:
        c.close()


def test_unit_kernel_lanczos_saturated_stars(argus):
    """Lanczos-3 through the unit kernel next to saturated star cores: units with masked AND bright pixels hand their
    sub-blocks to the FP64 stray kernel at run time; repeated calls on the cached plan give identical results (the
    run-time list is reset per call), value + weight and coadd forms."""
    from gpu_util import assert_coadd_matches, assert_values_match, coadd_oracle, gpu_resample_planned, oracle_reference, upload
    fr = _saturated_star_frame()
    c = argus.Context(0)
    try:
        c.set_fast_path(3)
        idx_or, _ = oracle.footprint(fr.wcs, 512, 512, fr.nside)
        d = upload(fr)
        vo, wo, fl = oracle_reference(fr, idx_or, "lanczos3")
        outs = []
        for _ in range(3):
            n, v, w = gpu_resample_planned(c, fr, d, "lanczos3")
            outs.append((v, w))
        assert_values_match(outs[0][0], outs[0][1], vo, wo, fl, "unit kernel, Lanczos-3, saturated stars")
        assert np.array_equal(outs[0][0], outs[2][0]) and np.array_equal(outs[0][1], outs[2][1])
        tiles = np.unique(idx_or >> 18)
        ppt = 1 << 18
        ref = coadd_oracle([fr] * 3, [idx_or] * 3, tiles, ppt, fr.nside, "lanczos3")
        s = torch.zeros(len(tiles) * ppt, dtype=torch.float32, device="cuda")
        ws = torch.zeros_like(s)
        for _ in range(3):
            argus.argus_resample_coadd(c, fr.wcs, 512, 512, fr.nside, "lanczos3", torch.from_numpy(tiles).cuda(), 256, s, ws, None, **d)
        torch.cuda.synchronize()
        argus.argus_plan_info(c)
        assert_coadd_matches(s.cpu().numpy(), ws.cpu().numpy(), ref, "unit kernel, Lanczos-3 coadd, same WCS three times")
    finally:
        c.close()


def test_resample_coadd_host_matches_device_path(argus, ctx, cfg0, cfg0_fp):
    """argus_resample_coadd_host (raw frame in HOST memory, pipelined uploads) accumulates exactly what
    argus_resample_coadd does from device memory, over several frames."""
    from gpu_util import upload
    d = upload(cfg0)
    tiles = torch.from_numpy(np.unique(cfg0_fp[0] >> 18)).cuda()
    n_slots = tiles.numel() << 18
    ref_s = torch.zeros(n_slots, dtype=torch.float32, device="cuda")
    ref_w = torch.zeros_like(ref_s)
    s = torch.zeros_like(ref_s)
    w = torch.zeros_like(ref_s)
    h_raw = torch.from_numpy(cfg0.raw).pin_memory()
    for _ in range(4):
        argus.argus_resample_coadd(ctx, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", tiles, 256, ref_s, ref_w, None, **d)
        argus.argus_resample_coadd_host(ctx, cfg0.wcs, 512, 512, cfg0.nside, "bilinear", h_raw, tiles, 256, s, w, None, bias=d["bias"],
                                        dark=d["dark"], flat=d["flat"], t_exp=cfg0.t_exp, sat_adu=cfg0.sat_adu, flat_min=cfg0.flat_min)
    argus.argus_host_wait(ctx)
    torch.cuda.synchronize()
    assert torch.equal(s, ref_s) and torch.equal(w, ref_w) and float(w.sum()) > 4 * 0.9 * len(cfg0_fp[0])
