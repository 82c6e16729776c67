"""GPU parity (-m gpu) of argus_segment_products against oracle/segments.py, through the C ABI.
Integer, byte and bit-pattern outputs (mini_id, mini_keep, n_mini, the binary16 segment data) are compared
bit-exactly; the FP32 weighted means within 1e-3 ADU + 1e-5 relative (north_star), the summed weights within
1e-5 relative (FP32 sums of at most 4^j terms against the fp64 sums)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import synth  # noqa: E402
from oracle import segments as oseg  # noqa: E402


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


def _run(argus, ctx, nside, nside_mini, idx, value, weight, targets, cap=None, tiles=None, nside_tile=None, stamp=True):
    dev = "cuda:0"
    n = idx.size
    cap = n if cap is None else cap
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    d = dict(mini_id=torch.full((cap,), -7, dtype=torch.int64, device=dev),
             mini_value=torch.full((cap,), float("nan"), dtype=torch.float32, device=dev),
             mini_weight=torch.full((cap,), float("nan"), dtype=torch.float32, device=dev),
             mini_keep=torch.full((cap,), 9, dtype=torch.uint8, device=dev) if stamp else None)
    n16 = n if tiles is None else tiles.size * (nside // nside_tile) ** 2
    seg16 = torch.zeros((n16,), dtype=torch.int16, device=dev) if tiles is not None else \
        torch.full((n16,), 0x5555, dtype=torch.int16, device=dev)
    nm = argus.argus_segment_products(ctx, nside, nside_mini, t(idx), t(value), t(weight), t(targets), seg16=seg16,
                                      tiles=None if tiles is None else t(tiles), nside_tile=nside_tile, **d)
    torch.cuda.synchronize()
    out = {k: (None if v is None else v.cpu().numpy()) for k, v in d.items()}
    out["seg16"] = seg16.cpu().numpy().view(np.uint16)
    out["n_mini"] = nm
    return out


def _compare(g, o, dense=False):
    nm = o["mini_id"].size
    assert g["n_mini"] == nm
    assert np.array_equal(g["mini_id"][:nm], o["mini_id"])
    if g["mini_keep"] is not None:
        assert np.array_equal(g["mini_keep"][:nm], o["mini_keep"])
    assert np.array_equal(g["seg16"], o["dense16"] if dense else o["seg16"])
    dw = np.abs(g["mini_weight"][:nm] - o["mini_weight"])
    assert np.all(dw <= 1e-5 * np.abs(o["mini_weight"]) + 1e-7), dw.max()
    ok = np.isfinite(o["mini_value"])
    dv = np.abs(g["mini_value"][:nm][ok].astype(np.float64) - o["mini_value"][ok])
    tol = 1e-3 + 1e-5 * np.abs(o["mini_value"][ok])
    assert np.all(dv <= tol), (dv / tol).max()
    assert np.array_equal(np.isnan(g["mini_value"][:nm]), np.isnan(o["mini_value"]))


@pytest.mark.parametrize("nside,nside_mini", [(1 << 17, 1 << 14), (1 << 17, 1 << 17), (1 << 18, 1 << 14), (1 << 12, 1 << 7)])
@pytest.mark.parametrize("n", [1, 63, 64, 65, 4095, 4096, 4097, 100003])
def test_segment_products_match_oracle(argus, ctx, nside, nside_mini, n):
    idx, value, weight = synth.footprint_like(1000 + n, 12 * nside * nside, n, run=max(64, (nside // nside_mini) ** 2 * 3))
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = synth.target_list(n, int(m[0]), int(m[-1]) + 1, 0.3)
    o = oseg.segment_products(idx, value, weight, nside, nside_mini, targets)
    g = _run(argus, ctx, nside, nside_mini, idx, value, weight, targets)
    _compare(g, o)
    if n == 100003 and nside_mini < nside:
        assert 0 < int(o["mini_keep"].sum()) < o["mini_keep"].size


def test_many_ctas_lookback_and_dense_footprint(argus, ctx):
    # 3.2 M pixels = 782 head-scan CTAs (look-back windows of 32); no holes: every minipix complete
    nside, nside_mini = 1 << 17, 1 << 14
    idx, value, weight = synth.footprint_like(5, 12 * nside * nside, 3_200_017, hole_frac=0.0, run=1 << 30)
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = synth.target_list(6, int(m[0]), int(m[-1]) + 1, 0.05)
    o = oseg.segment_products(idx, value, weight, nside, nside_mini, targets)
    g = _run(argus, ctx, nside, nside_mini, idx, value, weight, targets, cap=o["mini_id"].size)
    _compare(g, o)
    # and again with holes, twice in a row (scratch is reused; status words must be reset every call)
    idx, value, weight = synth.footprint_like(7, 12 * nside * nside, 1_000_003)
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = synth.target_list(8, int(m[0]), int(m[-1]) + 1, 0.5)
    o = oseg.segment_products(idx, value, weight, nside, nside_mini, targets)
    for _ in range(2):
        _compare(_run(argus, ctx, nside, nside_mini, idx, value, weight, targets), o)


def test_dense_tile_layout(argus, ctx):
    nside, nside_mini, nside_tile = 1 << 17, 1 << 14, 1 << 8        # the paper's NSIDE-256 segments: 2^18 px each
    idx, value, weight = synth.footprint_like(31, 12 * nside * nside, 700_001, run=50_000)
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = synth.target_list(32, int(m[0]), int(m[-1]) + 1, 0.4)
    tl = np.unique(idx >> 18)
    tiles = np.concatenate([tl[:1], tl[2:], [tl[-1] + 3]]).astype(np.int64) if tl.size > 2 else tl   # one absent, one unused
    o = oseg.segment_products(idx, value, weight, nside, nside_mini, targets, layout_tiles=tiles, nside_tile=nside_tile)
    g = _run(argus, ctx, nside, nside_mini, idx, value, weight, targets, tiles=tiles, nside_tile=nside_tile)
    _compare(g, o, dense=True)
    assert o["dense16"].any()
    # the same tiles as row-major 512 x 512 images (ARGUS_OPT_SEGMENT_RASTER)
    o_r = oseg.segment_products(idx, value, weight, nside, nside_mini, targets, layout_tiles=tiles, nside_tile=nside_tile, raster=True)
    assert not np.array_equal(o_r["dense16"], o["dense16"])
    ctx.set_segment_raster(True)
    try:
        g_r = _run(argus, ctx, nside, nside_mini, idx, value, weight, targets, tiles=tiles, nside_tile=nside_tile)
    finally:
        ctx.set_segment_raster(False)
    _compare(g_r, o_r, dense=True)


@pytest.mark.parametrize("raster", [False, True])
def test_dense_layout_with_large_and_small_minipix(argus, ctx, raster):
    # 1024-pixel minipix (generic path of the products kernel) and 4-pixel minipix, tiles of 64 x 64 pixels
    for nside, nside_mini, nside_tile in (((1 << 12), 1 << 7, 1 << 6), ((1 << 12), 1 << 11, 1 << 6)):
        idx, value, weight = synth.footprint_like(41 + nside_mini, 12 * nside * nside, 60_001, run=5000)
        m = oseg.minipix_of(idx, nside, nside_mini)
        targets = synth.target_list(42, int(m[0]), int(m[-1]) + 1, 0.5)
        tiles = np.unique(idx >> 12)[1:]
        o = oseg.segment_products(idx, value, weight, nside, nside_mini, targets, layout_tiles=tiles, nside_tile=nside_tile, raster=raster)
        ctx.set_segment_raster(raster)
        try:
            g = _run(argus, ctx, nside, nside_mini, idx, value, weight, targets, tiles=tiles, nside_tile=nside_tile)
        finally:
            ctx.set_segment_raster(False)
        _compare(g, o, dense=True)


def test_special_values_pack_bit_exactly(argus, ctx):
    nside, nside_mini = 1 << 17, 1 << 14
    v = np.array([0.0, -0.0, 1.0, 65504.0, 65519.99, 65520.0, 1e5, -1e5, np.inf, -np.inf, np.nan, 2.0 ** -24, 2.0 ** -25,
                  3 * 2.0 ** -25, 2.0 ** -14, 1 + 2.0 ** -11, 1 + 3 * 2.0 ** -11, 0.1, -1234.5, 6.1e-5, 5.9e-8, 1e-10],
                 dtype=np.float32)
    rng = np.random.default_rng(3)
    v = np.concatenate([v, (np.arange(2048) + 0.5).astype(np.float32) * np.float32(2.0 ** -24),
                        (10.0 ** rng.uniform(-9, 5, 20000) * rng.choice([-1, 1], 20000)).astype(np.float32)])
    idx = 64 * 777 + np.arange(v.size, dtype=np.int64)
    w = np.ones(v.size, np.float32)
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = np.unique(m)
    o = oseg.segment_products(idx, v, w, nside, nside_mini, targets)
    g = _run(argus, ctx, nside, nside_mini, idx, v, w, targets)
    assert np.array_equal(g["seg16"], o["seg16"])
    assert np.array_equal(g["mini_id"][:g["n_mini"]], o["mini_id"])
    # no stamping at all when mini_keep is not supplied
    g2 = _run(argus, ctx, nside, nside_mini, idx, v, w, np.zeros(0, np.int64), stamp=False)
    assert np.array_equal(g2["seg16"], oseg.pack_f16(v))


def test_top_of_the_index_range(argus, ctx):
    nside, nside_mini = 1 << 29, 1 << 26
    npix = 12 * nside * nside
    idx, value, weight = synth.footprint_like(9, npix, 20000, start=npix - 20000 * 3)
    idx = np.concatenate([idx[:-1], [npix - 1]])
    m = oseg.minipix_of(idx, nside, nside_mini)
    targets = synth.target_list(10, int(m[0]), int(m[-1]) + 1, 0.5)
    _compare(_run(argus, ctx, nside, nside_mini, idx, value, weight, targets),
             oseg.segment_products(idx, value, weight, nside, nside_mini, targets))


def test_count_only_capacity_async_and_errors(argus, ctx):
    dev = "cuda:0"
    nside, nside_mini = 1 << 17, 1 << 14
    idx, value, weight = synth.footprint_like(77, 12 * nside * nside, 50_000)
    o = oseg.segment_products(idx, value, weight, nside, nside_mini, np.zeros(0, np.int64))
    nm = o["mini_id"].size
    ti, tv, tw = (torch.from_numpy(a).to(dev) for a in (idx, value, weight))
    none = torch.zeros(0, dtype=torch.int64, device=dev)
    assert argus.argus_segment_products(ctx, nside, nside_mini, ti, tv, tw, none) == nm          # count only
    # capacity too small: error carries the required size, the first `cap` minipix are still right
    cap = nm // 2
    mid = torch.full((cap,), -1, dtype=torch.int64, device=dev)
    mv = torch.zeros(cap, dtype=torch.float32, device=dev)
    with pytest.raises(argus.ArgusError) as ei:
        argus.argus_segment_products(ctx, nside, nside_mini, ti, tv, tw, none, mini_id=mid, mini_value=mv)
    assert ei.value.status == -6 and "n_mini=%d" % nm in str(ei.value)
    assert np.array_equal(mid.cpu().numpy(), o["mini_id"][:cap])
    assert np.allclose(mv.cpu().numpy(), o["mini_value"][:cap], rtol=1e-5, atol=1e-3)
    # asynchronous form: count lands in a device scalar
    nd = torch.full((1,), -5, dtype=torch.int64, device=dev)
    mid = torch.full((nm,), -1, dtype=torch.int64, device=dev)
    assert argus.argus_segment_products(ctx, nside, nside_mini, ti, tv, tw, none, mini_id=mid, n_mini_dev=nd, sync=False) is None
    torch.cuda.synchronize()
    assert int(nd.item()) == nm and np.array_equal(mid.cpu().numpy(), o["mini_id"])
    # empty input
    e64, e32 = torch.zeros(0, dtype=torch.int64, device=dev), torch.zeros(0, dtype=torch.float32, device=dev)
    nd.fill_(-5)
    assert argus.argus_segment_products(ctx, nside, nside_mini, e64, e32, e32, none, n_mini_dev=nd) == 0
    assert int(nd.item()) == 0
    # argument errors
    for bad in ((nside, 3000), (nside, nside * 2), (3 << 10, 1 << 10)):
        with pytest.raises(argus.ArgusError) as ei:
            argus.argus_segment_products(ctx, bad[0], bad[1], ti, tv, tw, none)
        assert ei.value.status == -3
    with pytest.raises(argus.ArgusError) as ei:   # layout coarser than the minipix only
        argus.argus_segment_products(ctx, nside, 1 << 7, ti, tv, tw, none, mini_id=mid, tiles=torch.zeros(1, dtype=torch.int64, device=dev),
                                     nside_tile=1 << 8, seg16=torch.zeros(1 << 18, dtype=torch.int16, device=dev))
    assert ei.value.status == -2


def test_on_a_real_footprint(argus, ctx):
    """config 0 end to end: library footprint + fused resample -> segment products; oracle on the same arrays."""
    from gpu_util import upload
    fr = synth.config0()
    H, W = fr.shape
    d = upload(fr)
    n, idx = argus.argus_healpix_footprint(ctx, fr.wcs, W, H, fr.nside, want_indices=True)
    v = torch.empty(n, dtype=torch.float32, device="cuda:0")
    w = torch.empty(n, dtype=torch.float32, device="cuda:0")
    argus.argus_resample(ctx, fr.wcs, W, H, fr.nside, "bilinear", v, w, **d)
    torch.cuda.synchronize()
    idx_h, v_h, w_h = idx.cpu().numpy(), v.cpu().numpy(), w.cpu().numpy()
    m = oseg.minipix_of(idx_h, fr.nside, 1 << 14)
    targets = synth.target_list(4, int(m.min()), int(m.max()) + 1, 0.02)
    o = oseg.segment_products(idx_h, v_h, w_h, fr.nside, 1 << 14, targets)
    g = _run(argus, ctx, fr.nside, 1 << 14, idx_h, v_h, w_h, targets)
    _compare(g, o)
    assert 0 < o["mini_keep"].sum() < o["mini_keep"].size


def test_reduce_frame_host_equals_the_device_path(argus, ctx):
    """argus_reduce_frame_host (raw frame and products in HOST memory, pipelined) == argus_resample ->
    argus_healpix_footprint list -> argus_segment_products on device buffers, bit for bit, over several frames."""
    from gpu_util import upload
    fr = synth.config0()
    d = upload(fr)
    n, idx = argus.argus_healpix_footprint(ctx, fr.wcs, 512, 512, fr.nside)
    v = torch.empty(n, dtype=torch.float32, device="cuda")
    w = torch.empty_like(v)
    argus.argus_resample(ctx, fr.wcs, 512, 512, fr.nside, "bilinear", v, w, **d)
    none = torch.zeros(0, dtype=torch.int64, device="cuda")
    nm = argus.argus_segment_products(ctx, fr.nside, 1 << 14, idx, v, w, none)
    cap = nm + 7
    ref = dict(seg16=torch.empty(n, dtype=torch.int16, device="cuda"), mini_id=torch.empty(cap, dtype=torch.int64, device="cuda"),
               mini_value=torch.empty(cap, dtype=torch.float32, device="cuda"), mini_weight=torch.empty(cap, dtype=torch.float32, device="cuda"))
    assert argus.argus_segment_products(ctx, fr.nside, 1 << 14, idx, v, w, None, **ref) == nm
    torch.cuda.synchronize()
    h_raw = torch.from_numpy(fr.raw).pin_memory()
    outs = []
    for _ in range(4):
        o = dict(seg16_host=torch.zeros(n, dtype=torch.int16).pin_memory(), mini_id_host=torch.zeros(cap, dtype=torch.int64).pin_memory(),
                 mini_value_host=torch.zeros(cap, dtype=torch.float32).pin_memory(), mini_weight_host=torch.zeros(cap, dtype=torch.float32).pin_memory(),
                 n_mini_host=torch.zeros(1, dtype=torch.int64).pin_memory())
        argus.argus_reduce_frame_host(ctx, fr.wcs, 512, 512, fr.nside, "bilinear", n, h_raw, bias=d["bias"], dark=d["dark"], flat=d["flat"],
                                      t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min, **o)
        outs.append(o)
    argus.argus_host_wait(ctx)
    for o in outs:
        assert int(o["n_mini_host"].item()) == nm
        assert torch.equal(o["seg16_host"], ref["seg16"].cpu())
        assert torch.equal(o["mini_id_host"][:nm], ref["mini_id"].cpu()[:nm])
        assert torch.equal(o["mini_value_host"][:nm], ref["mini_value"].cpu()[:nm])
        assert torch.equal(o["mini_weight_host"][:nm], ref["mini_weight"].cpu()[:nm])
