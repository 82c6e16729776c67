"""Synthetic raw frames, calibration masters and WCS parameters (no method arithmetic).

See ``synth/__init__.py`` for the recipe and its citations.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import math

import numpy as np

#: PAPER.md:42 (Table 1) "Pixel Sampling 1.38 arcsec/pix".
PIXEL_SCALE_DEG = 1.38 / 3600.0
#: BASELINE.json configs[0]: FWHM 2.0 px Gaussian stars.
STAR_SIGMA_PX = 2.0 / 2.3548200450309493
FULL_W, FULL_H = 9576, 6388  # BASELINE.json configs[1]; "61 MPix"


@dataclass
class Wcs:
    """Sky->pixel WCS parameters ("one-directional mapping from
    celestial to pixel-plane coordinates").  Plain numbers only."""

    crval: tuple[float, float]  # deg (alpha0, delta0)
    crpix: tuple[float, float]  # 0-based px
    cd: tuple[tuple[float, float], tuple[float, float]]  # deg/px
    sip_order: int = 0
    ap: np.ndarray = field(default_factory=lambda: np.zeros(36))  # [p*6+q]
    bp: np.ndarray = field(default_factory=lambda: np.zeros(36))

    def as_array(self) -> np.ndarray:
        """Flat float64[81]: crval(2) crpix(2) cd(4, row-major) sip_order ap(36) bp(36)."""
        out = np.zeros(81, dtype=np.float64)
        out[0:2] = self.crval
        out[2:4] = self.crpix
        out[4:8] = (self.cd[0][0], self.cd[0][1], self.cd[1][0], self.cd[1][1])
        out[8] = float(self.sip_order)
        out[9:45] = self.ap
        out[45:81] = self.bp
        return out


@dataclass
class Frame:
    raw: np.ndarray  # uint16 [H][W]
    bias: np.ndarray  # float32 [H][W], ADU
    dark: np.ndarray  # float32 [H][W], ADU/s
    flat: np.ndarray  # float32 [H][W]
    bpm: np.ndarray | None  # uint8 [H][W] or None; non-zero = bad
    t_exp: float
    sat_adu: int
    flat_min: float
    wcs: Wcs
    nside: int
    kernel: str  # "bilinear" | "lanczos3"

    @property
    def shape(self) -> tuple[int, int]:
        return self.raw.shape  # (H, W)


def make_wcs(crval, crpix, rot_deg=0.0, scale_deg=PIXEL_SCALE_DEG, sip=None) -> Wcs:
    """CD = s * [[-cos r, sin r], [sin r, cos r]] (east-left, north-up at r = 0;
    SURVEY.md 8(c)-O4 reading of the silent paper)."""
    r = math.radians(rot_deg)
    cd = ((-scale_deg * math.cos(r), scale_deg * math.sin(r)),
          (scale_deg * math.sin(r), scale_deg * math.cos(r)))
    w = Wcs(crval=(float(crval[0]), float(crval[1])), crpix=(float(crpix[0]), float(crpix[1])), cd=cd)
    if sip is not None:
        w.sip_order, w.ap, w.bp = sip
    return w


def make_sip(rng: np.random.Generator, order: int = 3, half_axis_px: float = FULL_W / 2.0):
    """BASELINE.json configs[2]: "coefficients drawn N(0,1e-6) scaled per order".
    Reading: for n = p+q in {2..order}: sigma_n = 1e-6 * L^(2-n),
    L = half long axis in px; orders 0 and 1 are zero; AP then BP drawn in (p,q)
    lexicographic order."""
    ap = np.zeros(36)
    bp = np.zeros(36)
    for arr in (ap, bp):
        for p in range(order + 1):
            for q in range(order + 1 - p):
                n = p + q
                if n < 2:
                    continue
                arr[p * 6 + q] = rng.normal(0.0, 1e-6 * half_axis_px ** (2 - n))
    return order, ap, bp


def _scene(rng, W, H, n_stars, sky, fmin=1e2, fmax=1e6, stamp_r=8):
    """Sky + Gaussian stars sampled at pixel centres, in e-/px (float64 [H][W])."""
    sx = rng.uniform(-0.5, W - 0.5, n_stars)
    sy = rng.uniform(-0.5, H - 0.5, n_stars)
    q = rng.uniform(0.0, 1.0, n_stars)
    a, b = fmin ** -0.5, fmax ** -0.5
    flux = (a - q * (a - b)) ** -2.0  # inverse CDF of dN/dF ~ F^-1.5 on [fmin, fmax]
    scene = np.full((H, W), float(sky), dtype=np.float64)
    if n_stars == 0:
        return scene
    d = np.arange(-stamp_r, stamp_r + 1)
    cx = np.rint(sx).astype(np.int64)
    cy = np.rint(sy).astype(np.int64)
    px = cx[:, None, None] + d[None, None, :]  # [n,1,k]
    py = cy[:, None, None] + d[None, :, None]  # [n,k,1]
    r2 = (px - sx[:, None, None]) ** 2 + (py - sy[:, None, None]) ** 2
    amp = flux / (2.0 * math.pi * STAR_SIGMA_PX ** 2)
    val = amp[:, None, None] * np.exp(-0.5 * r2 / STAR_SIGMA_PX ** 2)
    px = np.broadcast_to(px, val.shape)
    py = np.broadcast_to(py, val.shape)
    ok = (px >= 0) & (px < W) & (py >= 0) & (py < H)
    np.add.at(scene.reshape(-1), (py[ok] * W + px[ok]), val[ok])
    return scene


def make_frame(seed: int, W: int, H: int, n_stars: int, wcs: Wcs, nside: int, kernel: str,
               t_exp: float = 30.0, sky: float = 200.0, masters=None, scene_seed=None) -> Frame:
    """BASELINE.json configs[0] noise/star/flat model (gain 1 e-/ADU so e- == ADU).
    ``scene_seed`` (configs[3]) draws the star field from its own generator so that
    consecutive exposures of one field share stars but not noise."""
    rng = np.random.Generator(np.random.PCG64(seed))
    srng = rng if scene_seed is None else np.random.Generator(np.random.PCG64(scene_seed))
    scene = _scene(srng, W, H, n_stars, sky)
    if masters is None:
        yy, xx = np.mgrid[0:H, 0:W]
        r2 = ((xx - (W - 1) / 2.0) ** 2 + (yy - (H - 1) / 2.0) ** 2) / (((W - 1) / 2.0) ** 2 + ((H - 1) / 2.0) ** 2)
        del yy, xx
        flat = (1.0 - 0.1 * r2) * (1.0 + rng.normal(0.0, 0.01, (H, W)))
        del r2
        flat = flat.astype(np.float32)
        bias = np.full((H, W), 1000.0, dtype=np.float32)
        dark = np.full((H, W), 0.005, dtype=np.float32)
    else:
        bias, dark, flat = masters
    signal = rng.normal(0.0, 1.7, (H, W))
    signal += 1000.0
    scene *= flat
    signal += rng.poisson(scene)
    del scene
    signal += rng.poisson(0.005 * t_exp, (H, W))
    raw = np.clip(np.rint(signal), 0, 65535).astype(np.uint16)
    return Frame(raw=raw, bias=bias, dark=dark, flat=flat, bpm=None, t_exp=float(t_exp),
                 sat_adu=65535, flat_min=0.1, wcs=wcs, nside=int(nside), kernel=kernel)


def inject_defects(fr: Frame) -> Frame:
    """Mask-logic parity frame: a saturated 9x9 block, a bad-pixel
    column, a flat < flat_min patch, one NaN flat pixel."""
    H, W = fr.shape
    raw = fr.raw.copy()
    flat = fr.flat.copy()
    bpm = np.zeros((H, W), dtype=np.uint8)
    y0, x0 = H // 3, W // 3
    raw[y0:y0 + 9, x0:x0 + 9] = 65535
    bpm[:, (2 * W) // 3] = 1
    flat[H // 2:H // 2 + 12, W // 5:W // 5 + 7] = 0.05
    flat[H // 4, W // 2] = np.nan
    return Frame(raw=raw, bias=fr.bias, dark=fr.dark, flat=flat, bpm=bpm, t_exp=fr.t_exp,
                 sat_adu=fr.sat_adu, flat_min=fr.flat_min, wcs=fr.wcs, nside=fr.nside, kernel=fr.kernel)


# ----------------------------------------------------------------------------- configs
def config0(seed: int = 0, kernel: str = "bilinear") -> Frame:
    """BASELINE.json configs[0]: 512x512, 300 stars, CRVAL (30,+20), nside 2^17."""
    W = H = 512
    wcs = make_wcs((30.0, 20.0), ((W - 1) / 2.0, (H - 1) / 2.0), 0.0)
    return make_frame(seed, W, H, 300, wcs, 1 << 17, kernel)


def config1(seed: int = 1, kernel: str = "bilinear", W: int = FULL_W, H: int = FULL_H) -> Frame:
    """BASELINE.json configs[1]: one full IMX455 frame, ~60k stars, 0.3 deg rotation."""
    wcs = make_wcs((30.0, 20.0), ((W - 1) / 2.0, (H - 1) / 2.0), 0.3)
    n_stars = int(round(60000 * (W * H) / float(FULL_W * FULL_H)))
    return make_frame(seed, W, H, n_stars, wcs, 1 << 17, kernel)


def config2_wcs(k: int, W: int = FULL_W, H: int = FULL_H) -> Wcs:
    """BASELINE.json configs[2]: 38 pointings over dec -20..+72, SIP order 3."""
    rng = np.random.Generator(np.random.PCG64(100 + k + 10_000))
    dec = -20.0 + 92.0 * k / 37.0
    ra = (137.508 * k) % 360.0
    rot = rng.uniform(-1.0, 1.0)
    sip = make_sip(rng, 3, W / 2.0)
    return make_wcs((ra, dec), ((W - 1) / 2.0, (H - 1) / 2.0), rot, sip=sip)


def config2_frame(k: int, W: int = FULL_W, H: int = FULL_H) -> Frame:
    wcs = config2_wcs(k, W, H)
    n_stars = int(round(60000 * (W * H) / float(FULL_W * FULL_H)))
    return make_frame(100 + k, W, H, n_stars, wcs, 1 << 17, "lanczos3")


def config3_frame(k: int, W: int = FULL_W, H: int = FULL_H, masters=None) -> Frame:
    """BASELINE.json configs[3]: 1 s exposures, sky 7 e-/px, +-0.5 px dither, shared masters."""
    rng = np.random.Generator(np.random.PCG64(300 + k + 10_000))
    dx, dy = rng.uniform(-0.5, 0.5, 2)
    wcs = make_wcs((30.0, 20.0), ((W - 1) / 2.0 + dx, (H - 1) / 2.0 + dy), 0.3)
    n_stars = int(round(60000 * (W * H) / float(FULL_W * FULL_H)))
    # same star field every frame (scene_seed), own noise realisation per frame (seed)
    return make_frame(300 + k, W, H, n_stars, wcs, 1 << 17, "bilinear", t_exp=1.0, sky=7.0,
                      masters=masters, scene_seed=3000)


def config4_frame(k: int, W: int = FULL_W, H: int = FULL_H) -> Frame:
    """BASELINE.json configs[4]: 3x3 mosaic around (30,+20), SIP order 3, nside 2^18, Lanczos-3."""
    rng = np.random.Generator(np.random.PCG64(400 + k + 10_000))
    i, j = k % 3 - 1, k // 3 - 1
    dec = 20.0 + 2.3 * j
    ra = 30.0 + 3.5 * i / math.cos(math.radians(dec))
    sip = make_sip(rng, 3, W / 2.0)
    wcs = make_wcs((ra, dec), ((W - 1) / 2.0, (H - 1) / 2.0), rng.uniform(-1.0, 1.0), sip=sip)
    n_stars = int(round(60000 * (W * H) / float(FULL_W * FULL_H)))
    return make_frame(400 + k, W, H, n_stars, wcs, 1 << 18, "lanczos3")


def special_pointings() -> dict[str, tuple[tuple[float, float], float, int]]:
    """Parity-only pointings: name -> (crval deg, rotation deg, nside)."""
    ring = math.degrees(math.asin(2.0 / 3.0))  # |dec| of the belt/cap ring, 41.8103 deg
    return {
        "belt_cap_ring": ((100.0, ring), 10.0, 1 << 17),
        "belt_cap_ring_south": ((200.0, -ring), -20.0, 1 << 17),
        "face_edge_belt": ((90.0, 10.0), 5.0, 1 << 17),
        "four_face_corner": ((45.0, 0.0), 0.0, 1 << 17),
        "ra_wrap": ((0.0, -5.0), 33.0, 1 << 17),
        "north_pole": ((123.0, 89.9), 0.0, 1 << 17),
        "south_cap": ((300.0, -60.0), 45.0, 1 << 17),
        "nside_2p18": ((30.0, 20.0), 0.3, 1 << 18),
        "cap_face_edge": ((90.0, 60.0), 15.0, 1 << 17),
    }
