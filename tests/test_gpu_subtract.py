"""GPU parity (-m gpu) of argus_subtract_tiles (direct image subtraction per tile) against
oracle/subtract.py, through the C ABI, on identical float32 (sum, wsum) inputs.

Tolerances: alpha, beta to 1e-6 relative (FP64 sums of float32 images in a different order);
n_valid exact; the difference to north_star's value tolerance applied to its operands, 1e-3 + 1e-5 max(|s|, |alpha r +
beta|) (float32 quotients, one fma, one subtraction); the significance to that tolerance divided by sigma + 1e-5 |S|.
Detection is a floating-point decision: the oracle reports the margins (threshold, local maximum); candidates with
margins above the tolerance must be found, records found must have margins above minus the tolerance."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import synth  # noqa: E402
from oracle import subtract as osub  # noqa: E402

DEV = "cuda:0"


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


def gpu_subtract(argus, ctx, tiles, nside_tile, nside, arrs, cap=100000, want_sig=True, **kw):
    t = torch.from_numpy(np.asarray(tiles, dtype=np.int64)).to(DEV)
    d = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(DEV) for a in arrs]
    n = d[0].numel()
    diff = torch.full((n,), float("nan"), dtype=torch.float32, device=DEV)
    sig = torch.full((n,), float("nan"), dtype=torch.float32, device=DEV) if want_sig else None
    al = torch.full((len(tiles),), float("nan"), dtype=torch.float32, device=DEV)
    be = torch.full_like(al, float("nan"))
    nv = torch.full((len(tiles),), -1, dtype=torch.int32, device=DEV)
    out = torch.zeros(cap * 32, dtype=torch.uint8, device=DEV)
    n_dev = torch.full((1,), -1, dtype=torch.int64, device=DEV)
    k = argus.argus_subtract_tiles(ctx, t, nside_tile, nside, d[0], d[1], d[2], d[3], diff, sig, out, alpha_out=al, beta_out=be,
                                   nvalid_out=nv, n_dev=n_dev, **kw)
    assert int(n_dev.item()) == k
    rec = out.cpu().numpy()[:k * 32].view(argus.TRANSIENT_DTYPE)
    return dict(diff=diff.cpu().numpy(), sig=None if sig is None else sig.cpu().numpy(), alpha=al.cpu().numpy(), beta=be.cpu().numpy(),
                n_valid=nv.cpu().numpy(), rec=rec)


def compare(g, tiles, ppt, nside, arrs, max_ambiguous=3, **kw):
    a32 = [np.ascontiguousarray(a, dtype=np.float32) for a in arrs]
    okw = dict(kw)
    okw["match"] = {"none": osub.MATCH_NONE, "affine": osub.MATCH_AFFINE}[kw.get("match", "affine")]
    o = osub.subtract_tiles(tiles, ppt, nside, *a32, slack=0.5, **okw)
    n_tiles = len(tiles)
    assert np.array_equal(g["n_valid"], o["n_valid"])
    assert np.all(np.abs(g["alpha"] - o["alpha"]) <= 1e-6 * np.abs(o["alpha"]) + 1e-7)
    assert np.all(np.abs(g["beta"] - o["beta"]) <= 1e-6 * np.abs(o["beta"]) + 1e-4 * np.abs(o["alpha"]) + 1e-5)
    sw, rw = a32[1].astype(np.float64), a32[3].astype(np.float64)
    valid = (sw >= kw.get("sci_wmin", 0.5)) & (rw >= kw.get("ref_wmin", 0.5))
    with np.errstate(all="ignore"):
        s = np.where(valid, a32[0] / np.where(valid, sw, 1), 0.0)
        m = np.where(valid, np.repeat(o["alpha"], ppt) * (a32[2] / np.where(valid, rw, 1)) + np.repeat(o["beta"], ppt), 0.0)
    tol_d = 1e-3 + 1e-5 * np.maximum(np.abs(s), np.abs(m))
    dd = np.abs(g["diff"] - o["diff"])
    assert np.all(dd <= tol_d), "difference off by %.3f x tolerance" % (dd / tol_d).max()
    assert np.all(g["diff"][~valid] == 0)
    rn, gain = kw.get("read_noise", 1.7), kw.get("gain", 1.0)
    with np.errstate(all="ignore"):
        sigma = np.sqrt((rn ** 2 + np.maximum(m, 0) / gain) * (1.0 / np.where(valid, sw, 1) + np.repeat(o["alpha"], ppt) ** 2 / np.where(valid, rw, 1)))
    tol_s = tol_d / sigma + 1e-5 * np.abs(o["sig"])
    if g["sig"] is not None:
        ds = np.abs(g["sig"] - o["sig"])
        assert np.all(ds[valid] <= tol_s[valid]), "significance off by %.3f x tolerance" % (ds[valid] / tol_s[valid]).max()
        assert np.all(g["sig"][~valid] == 0)
    # catalogue by decision margins
    c = o["cat"]
    slot_of = lambda pix: np.searchsorted(tiles, pix // ppt) * ppt + pix % ppt
    eps = tol_s[slot_of(c["pixel"])] if c["pixel"].size else np.zeros(0)
    must = c["strict"] & (c["m_thr"] > eps) & (c["m_max"] > 2 * eps)
    may = (c["m_thr"] > -eps) & (c["m_max"] > -2 * eps)
    rec = g["rec"]
    assert np.all(np.diff(rec["pixel"]) > 0), "catalogue not in ascending nested order (R-X8)"
    assert np.isin(c["pixel"][must], rec["pixel"]).all(), "a clear candidate is missing"
    assert np.isin(rec["pixel"], c["pixel"][may]).all(), "a record is not a candidate"
    n_amb = int((may & ~must).sum())
    assert n_amb <= max(max_ambiguous, 2e-3 * max(int(must.sum()), 1)), "%d ambiguous decisions" % n_amb
    pos = {int(p): i for i, p in enumerate(c["pixel"].tolist())}
    j = np.array([pos[int(p)] for p in rec["pixel"].tolist()], dtype=np.int64)
    if j.size:
        e = eps[j]
        td = tol_d[slot_of(rec["pixel"])]
        assert np.all(np.abs(rec["sig"] - c["sig"][j]) <= e) and np.all(np.abs(rec["diff"] - c["diff"][j]) <= td)
        assert np.all(np.abs(rec["flux"] - c["flux"][j]) <= 9 * td) and np.all(np.abs(rec["noise"] - c["noise"][j]) <= 1e-5 * c["noise"][j])
        assert np.array_equal(rec["tile_rank"], c["tile_rank"][j])
    return int(must.sum()), n_amb


def synth_pairs(seed, n_tiles, side, n_src=6, mask_frac=0.03, alpha=0.93, beta=4.0, ref_frames=30.0):
    """Tile-dense (sum, wsum) pairs: a smooth sky + stars reference (weight ~ ref_frames), a noisy scaled science frame
    with weights in {0, 0.5 .. 1}, masked pixels in both, and injected point sources (also at tile edges and corners)."""
    rng = np.random.default_rng(seed)
    ppt = side * side
    out = [np.zeros(n_tiles * ppt) for _ in range(4)]
    y, x = np.mgrid[0:side, 0:side]
    for t in range(n_tiles):
        r = 200.0 + 0.3 * x - 0.2 * y
        for _ in range(8):
            cx, cy, a = rng.uniform(0, side), rng.uniform(0, side), rng.uniform(100, 20000)
            r = r + a * np.exp(-((x - cx) ** 2 + (y - cy) ** 2) / (2 * 0.9 ** 2))
        s = alpha * r + beta + rng.normal(0, 1.0, r.shape) * np.sqrt(1.7 ** 2 + np.maximum(alpha * r + beta, 0))
        pts = [(0, 0), (side - 1, side - 1), (0, side // 2)] + [tuple(rng.integers(0, side, 2)) for _ in range(n_src)]
        for (py, px) in pts:
            s[py, px] += rng.uniform(150, 600)
        ws = np.where(rng.random(r.shape) < mask_frac, 0.0, np.where(rng.random(r.shape) < 0.05, rng.uniform(0.3, 1.0, r.shape), 1.0))
        wr = np.where(rng.random(r.shape) < mask_frac, 0.0, ref_frames * rng.uniform(0.8, 1.0, r.shape))
        sl = slice(t * ppt, (t + 1) * ppt)
        out[0][sl] = osub.grid_to_tile(s * ws); out[1][sl] = osub.grid_to_tile(ws)
        out[2][sl] = osub.grid_to_tile(r * wr); out[3][sl] = osub.grid_to_tile(wr)
    return out


@pytest.mark.parametrize("side_log2,n_tiles", [(5, 3), (6, 2), (7, 2)])
@pytest.mark.parametrize("match", ["affine", "none"])
def test_synthetic_tiles(argus, ctx, side_log2, n_tiles, match):
    nside = 1 << 12
    nside_tile = nside >> side_log2
    side = 1 << side_log2
    tiles = np.array([5, 77, 1000][:n_tiles], dtype=np.int64)
    arrs = synth_pairs(10 + side_log2, n_tiles, side, alpha=0.93 if match == "affine" else 1.0, beta=4.0 if match == "affine" else 0.0)
    kw = dict(match=match, k_sigma=5.0, read_noise=1.7, gain=1.0)
    g = gpu_subtract(argus, ctx, tiles, nside_tile, nside, arrs, **kw)
    n_must, n_amb = compare(g, tiles, side * side, nside, arrs, **kw)
    assert n_must >= 3 * n_tiles
    print("subtract side %d %s: %d records, %d clear, %d ambiguous, alpha %s" % (side, match, g["rec"].size, n_must, n_amb, g["alpha"]))


def test_fit_fallbacks_and_parameters(argus, ctx):
    nside, nside_tile, side = 1 << 12, 1 << 7, 32
    ppt = side * side
    tiles = np.array([1, 2, 3], dtype=np.int64)
    arrs = synth_pairs(3, 3, side)
    arrs[1][:ppt] = 0.0                              # tile 0: no valid pixel
    arrs[1][ppt + 10:2 * ppt] = 0.0                  # tile 1: 10 valid pixels at most (< n_min)
    arrs[2][2 * ppt:] = 300.0 * arrs[3][2 * ppt:]    # tile 2: constant reference
    kw = dict(match="affine", n_min=16, sci_wmin=0.4, ref_wmin=2.0, read_noise=2.5, gain=0.7, k_sigma=3.0)
    g = gpu_subtract(argus, ctx, tiles, nside_tile, nside, arrs, **kw)
    compare(g, tiles, ppt, nside, arrs, max_ambiguous=6, **kw)
    assert g["n_valid"][0] == 0 and g["alpha"][0] == 1 and g["beta"][0] == 0 and g["n_valid"][1] <= 10 and g["alpha"][1] == 1
    assert g["alpha"][2] == 1
    # without the optional outputs, count only, capacity error
    t = torch.from_numpy(tiles).to(DEV)
    d = [torch.from_numpy(a.astype(np.float32)).to(DEV) for a in arrs]
    diff = torch.empty_like(d[0])
    n = argus.argus_subtract_tiles(ctx, t, nside_tile, nside, *d, diff, None, None, **kw)
    assert n == g["rec"].size and np.array_equal(diff.cpu().numpy(), g["diff"])
    small = torch.zeros(2 * 32, dtype=torch.uint8, device=DEV)
    with pytest.raises(argus.ArgusError) as e:
        argus.argus_subtract_tiles(ctx, t, nside_tile, nside, *d, diff, None, small, **kw)
    assert e.value.status == -6 and ("n_candidates=%d" % n) in str(e.value)
    with pytest.raises(argus.ArgusError):
        argus.argus_subtract_tiles(ctx, t, nside_tile, nside, *d, diff, None, None, read_noise=0.0)
    # empty layout
    z = torch.zeros(0, dtype=torch.float32, device=DEV)
    assert argus.argus_subtract_tiles(ctx, torch.zeros(0, dtype=torch.int64, device=DEV), nside_tile, nside, z, z, z, z, z, None, None) == 0


def _coadd_pair(argus, ctx, frames, tiles_dev, nside, n_slots):
    from gpu_util import upload
    s = torch.zeros(n_slots, dtype=torch.float32, device=DEV)
    w = torch.zeros_like(s)
    for f in frames:
        argus.argus_resample_coadd(ctx, f.wcs, f.shape[1], f.shape[0], nside, "bilinear", tiles_dev, 256, s, w, None, **upload(f))
    torch.cuda.synchronize()
    return s, w


def test_end_to_end_injected_transient(argus, ctx):
    """The paper's flow (Fig. 3 :169): reference = coadd of earlier frames on the HEALPix grid, science =
    the next frame with a transient injected into its raw pixels; argus_resample_coadd produces both pairs, then the
    subtraction.  Parity with the oracle on the pairs the GPU produced; the transient is among the candidates."""
    W = H = 512
    nside = 1 << 17
    # nine 1 s exposures of ONE sky (configs[3] recipe: sky 7 e-/px, shared star field and masters) on one WCS: the
    # synthetic star field is fixed in detector coordinates, so a dithered WCS would move it on the sky
    wcs = synth.make_wcs((30.0, 20.0), (255.5, 255.5), 0.3)
    frames = [synth.make_frame(300 + k, W, H, 257, wcs, nside, "bilinear", t_exp=1.0, sky=7.0, scene_seed=3000) for k in range(9)]
    sci = frames[8]
    raw = sci.raw.astype(np.float64)
    yy, xx = np.mgrid[0:H, 0:W]
    tx, ty = 301.3, 207.6
    raw += 120.0 * np.exp(-0.5 * ((xx - tx) ** 2 + (yy - ty) ** 2) / 0.85 ** 2)
    sci.raw = np.clip(np.rint(raw), 0, 65535).astype(np.uint16)
    fps = [oracle.footprint(wcs, W, H, nside)[0]]
    tiles = np.unique(fps[0] >> 18)
    ppt = 1 << 18
    td = torch.from_numpy(tiles).to(DEV)
    rs, rw = _coadd_pair(argus, ctx, frames[:8], td, nside, len(tiles) * ppt)
    ss, sw = _coadd_pair(argus, ctx, [sci], td, nside, len(tiles) * ppt)
    arrs = [a.cpu().numpy() for a in (ss, sw, rs, rw)]
    kw = dict(match="affine", k_sigma=5.0, read_noise=1.7, gain=1.0, ref_wmin=2.0)
    g = gpu_subtract(argus, ctx, tiles, 256, nside, arrs, **kw)
    n_must, n_amb = compare(g, tiles, ppt, nside, arrs, max_ambiguous=6, **kw)
    # the injected source: the HEALPix pixel nearest to its detector position
    x, y, _ = oracle.pix2xy(sci.wcs, nside, g["rec"]["pixel"])
    dist = np.hypot(x - tx, y - ty)
    assert dist.min() < 1.0 and g["rec"]["sig"][dist.argmin()] > 10
    assert g["rec"].size <= 3                      # the transient and at most a noise peak or two at 5 sigma
    assert np.all(np.abs(g["alpha"] - 1) < 0.05) and np.all(np.abs(g["beta"]) < 0.5)
    print("end to end: %d candidates (%d clear, %d ambiguous), transient S = %.1f, flux %.0f" % (g["rec"].size, n_must, n_amb,
          g["rec"]["sig"][dist.argmin()], g["rec"]["flux"][dist.argmin()]))
