"""Pins S1-S5 for oracle/segments.py (segment products): each checks the oracle against
something other than itself -- Python's own binary16 encoder and hand-derived bit patterns, the HEALPix
geometry (a child's centre lies in its parent), closed forms, conservation laws and pure-Python brute force."""
import struct

import numpy as np
import pytest

import oracle
from oracle import segments as seg


def _py_half_bits(x):
    return struct.unpack("<H", struct.pack("<e", x))[0]


def test_s1_pack_f16_hand_values():
    # (value, bits): binary16 = 1 sign, 5 exponent (bias 15), 10 fraction bits; ties go to the even fraction.
    cases = [
        (0.0, 0x0000), (-0.0, 0x8000), (1.0, 0x3C00), (-2.0, 0xC000), (0.5, 0x3800),
        (65504.0, 0x7BFF),                 # largest finite
        (65519.99, 0x7BFF),                # below the halfway point to 65536: rounds down
        (1.0e5, 0x7BFF), (-1.0e5, 0xFBFF),  # reading R-S2: clamped, not infinity
        (float("inf"), 0x7BFF), (float("-inf"), 0xFBFF),
        (2.0 ** -24, 0x0001),              # smallest subnormal
        (2.0 ** -25, 0x0000),              # tie between 0 and 2^-24: even -> 0
        (3 * 2.0 ** -25, 0x0002),          # tie between 1 and 2 (x 2^-24): even -> 2
        (2.0 ** -14, 0x0400),              # smallest normal
        (1.0 + 2.0 ** -11, 0x3C00),        # tie: even -> 1.0
        (1.0 + 3 * 2.0 ** -11, 0x3C02),    # tie: even -> 1 + 2 ulp
        (1.0 + 2.0 ** -11 + 2.0 ** -20, 0x3C01),  # just above the tie: rounds up
        (0.1, 0x2E66), (1000.0, 0x63D0), (-1234.5, 0xE4D2),
    ]
    v = np.array([c[0] for c in cases], dtype=np.float32)
    got = seg.pack_f16(v)
    for (x, want), g in zip(cases, got):
        assert int(g) == want, (x, hex(int(g)), hex(want))
    assert int(seg.pack_f16(np.array([np.nan], np.float32))[0]) == 0x7E00
    assert int(seg.pack_f16(np.array([-np.nan], np.float32))[0]) == 0x7E00


def test_s1_pack_f16_matches_python_struct_encoder():
    rng = np.random.default_rng(5)
    v = np.concatenate([
        rng.normal(0, 1, 4000), rng.normal(1000, 300, 4000), rng.uniform(-65504, 65504, 4000),
        10.0 ** rng.uniform(-9, 4.8, 4000) * rng.choice([-1, 1], 4000),
        (np.arange(2048) + 0.5) * 2.0 ** -24,        # every subnormal tie
        1024.0 + np.arange(4096) * 0.25,              # ulp = 1 here: exact quarters, halves are ties
    ]).astype(np.float32)
    v = v[np.abs(v) <= 65504.0]
    got = seg.pack_f16(v)
    want = np.array([_py_half_bits(float(x)) for x in v], dtype=np.uint16)
    assert np.array_equal(got, want)


@pytest.mark.parametrize("nside,nside_mini", [(1 << 17, 1 << 14), (1 << 18, 1 << 14), (64, 8), (32, 32)])
def test_s2_minipix_is_the_pixel_that_contains_the_child_centre(nside, nside_mini):
    # geometry, not bit arithmetic: centre of p (pix2ang at nside) located at nside_mini by ang2pix
    rng = np.random.default_rng(11)
    npix = 12 * nside * nside
    p = np.unique(np.concatenate([rng.integers(0, npix, 3000), [0, npix - 1],
                                  np.arange(12) * nside * nside, np.arange(1, 13) * nside * nside - 1]))
    got = seg.minipix_of(p, nside, nside_mini)
    for pi, gi in zip(p, got):
        th, ph = oracle.pix2ang(nside, int(pi))
        assert oracle.ang2pix(nside_mini, th, ph) == int(gi)


def test_s2_every_minipix_has_4_pow_j_children():
    nside, nside_mini = 16, 2
    m = seg.minipix_of(np.arange(12 * nside * nside), nside, nside_mini)
    ids, cnt = np.unique(m, return_counts=True)
    assert np.array_equal(ids, np.arange(12 * nside_mini * nside_mini))
    assert np.all(cnt == (nside // nside_mini) ** 2)
    assert np.all(np.diff(m) >= 0)         # children of one minipix are consecutive nested indices


def _random_footprint(rng, nside, n, holes=True):
    npix = 12 * nside * nside
    start = int(rng.integers(0, npix - 4 * n))
    idx = start + np.arange(2 * n, dtype=np.int64)
    if holes:
        idx = idx[rng.random(idx.size) < 0.7]
    idx = idx[:n]
    value = rng.normal(1200, 400, idx.size).astype(np.float32)
    weight = np.where(rng.random(idx.size) < 0.1, 0.0, rng.uniform(0.5, 1.0, idx.size)).astype(np.float32)
    return idx, value, weight


def test_s3_lowres_brute_force_and_conservation():
    rng = np.random.default_rng(3)
    nside, nside_mini = 256, 32
    idx, value, weight = _random_footprint(rng, nside, 5000)
    r = seg.segment_products(idx, value, weight, nside, nside_mini, targets=[])
    # brute force with Python containers and Fractions-free exact-enough double sums in pixel order
    acc = {}
    for p, v, w in zip(idx.tolist(), value.tolist(), weight.tolist()):
        s = acc.setdefault(p // 64, [0.0, 0.0])
        s[0] += w
        s[1] += w * v
    assert sorted(acc) == r["mini_id"].tolist()
    for k, mid in enumerate(r["mini_id"].tolist()):
        sw, swv = acc[mid]
        assert r["mini_weight"][k] == pytest.approx(sw, rel=1e-13, abs=1e-13)
        assert r["mini_value"][k] == pytest.approx(swv / sw if sw else 0.0, rel=1e-12, abs=1e-12)
    # conservation: the weighted flux of the low-resolution map is that of the input
    tot = float(np.sum(weight.astype(np.float64) * value.astype(np.float64)))
    assert float(np.sum(r["mini_weight"] * r["mini_value"])) == pytest.approx(tot, rel=1e-12)
    assert float(np.sum(r["mini_weight"])) == pytest.approx(float(np.sum(weight.astype(np.float64))), rel=1e-13)


def test_s3_lowres_closed_forms():
    nside, nside_mini = 1 << 17, 1 << 14
    base = 7 * 64 * 12345
    idx = base + np.arange(3 * 64, dtype=np.int64)
    # constant image -> the same constant, whatever the weights; zero total weight -> 0
    w = np.concatenate([np.linspace(0.5, 1, 64), np.zeros(64), np.ones(64)]).astype(np.float32)
    r = seg.segment_products(idx, np.full(idx.size, 321.5, np.float32), w, nside, nside_mini, targets=[])
    assert r["mini_id"].tolist() == [base // 64, base // 64 + 1, base // 64 + 2]
    assert r["mini_value"].tolist() == pytest.approx([321.5, 0.0, 321.5], rel=1e-14)
    assert r["mini_weight"].tolist() == pytest.approx([float(np.sum(w[:64].astype(np.float64))), 0.0, 64.0], rel=1e-14)
    # unit weights, value = offset in the minipix -> arithmetic mean (0 + ... + 63) / 64 = 31.5
    v = np.tile(np.arange(64, dtype=np.float32), 3)
    r = seg.segment_products(idx, v, np.ones(idx.size, np.float32), nside, nside_mini, targets=[])
    assert r["mini_value"].tolist() == pytest.approx([31.5] * 3, rel=1e-14)
    # one pixel of weight 1 among zeros -> that pixel's value
    w = np.zeros(idx.size, np.float32)
    w[[5, 64 + 63, 128]] = 1
    r = seg.segment_products(idx, v, w, nside, nside_mini, targets=[])
    assert r["mini_value"].tolist() == pytest.approx([5.0, 63.0, 0.0], abs=1e-14)


def test_s3_lowres_is_associative_over_levels():
    # weighted means compose: 8x in one step == 2x three times with the summed weights carried along
    rng = np.random.default_rng(8)
    nside = 1 << 12
    idx, value, weight = _random_footprint(rng, nside, 20000)
    one = seg.segment_products(idx, value, weight, nside, nside >> 3, targets=[])
    ids, v, w = idx, value.astype(np.float64), weight.astype(np.float64)
    ns = nside
    for _ in range(3):
        r = seg.segment_products(ids, v, w, ns, ns >> 1, targets=[])
        ids, v, w, ns = r["mini_id"], r["mini_value"], r["mini_weight"], ns >> 1
    assert np.array_equal(ids, one["mini_id"])
    assert np.allclose(w, one["mini_weight"], rtol=1e-12, atol=0)
    assert np.allclose(v, one["mini_value"], rtol=1e-11, atol=1e-11)


def test_s4_stamping_against_python_sets():
    rng = np.random.default_rng(21)
    nside, nside_mini = 1 << 17, 1 << 14
    idx, value, weight = _random_footprint(rng, nside, 30000)
    minis = sorted(set((idx // 64).tolist()))
    chosen = set(rng.choice(minis, len(minis) // 5, replace=False).tolist())
    foreign = {minis[0] - 3, minis[-1] + 10, 0, 12 * nside_mini ** 2 - 1} - set(minis)
    targets = np.array(sorted(chosen | foreign) + list(chosen)[:7], dtype=np.int64)   # duplicates allowed
    r = seg.segment_products(idx, value, weight, nside, nside_mini, targets)
    assert r["mini_id"].tolist() == minis
    assert r["mini_keep"].tolist() == [1 if m in chosen else 0 for m in minis]
    want = [(_py_half_bits(float(v)) if (p // 64) in chosen else 0) for p, v in zip(idx.tolist(), value.tolist())]
    assert r["seg16"].tolist() == want
    # all minipix are targets -> plain packing; none -> all zero
    allr = seg.segment_products(idx, value, weight, nside, nside_mini, np.array(minis))
    assert np.array_equal(allr["seg16"], seg.pack_f16(value)) and np.all(allr["mini_keep"] == 1)
    none = seg.segment_products(idx, value, weight, nside, nside_mini, np.zeros(0, np.int64))
    assert not none["seg16"].any() and not none["mini_keep"].any()
    # stamping does not touch the low-resolution map (low-resolution maps cover the whole sky)
    assert np.array_equal(none["mini_value"], allr["mini_value"])


def test_s5_dense_tile_layout_brute_force():
    rng = np.random.default_rng(2)
    nside, nside_mini, nside_tile = 1 << 10, 1 << 7, 1 << 5      # ppt = 32^2 = 1024
    idx, value, weight = _random_footprint(rng, nside, 6000)
    tiles_all = sorted(set((idx // 1024).tolist()))
    tiles = np.array([t for k, t in enumerate(tiles_all) if k != 1] + [tiles_all[-1] + 5], dtype=np.int64)  # one absent, one unused
    targets = np.unique(idx // 64)[::2]
    r = seg.segment_products(idx, value, weight, nside, nside_mini, targets, layout_tiles=tiles, nside_tile=nside_tile)
    dense = np.zeros(tiles.size * 1024, np.uint16)
    tl = tiles.tolist()
    for p, b in zip(idx.tolist(), r["seg16"].tolist()):
        if p // 1024 in tl:
            dense[tl.index(p // 1024) * 1024 + p % 1024] = b
    assert np.array_equal(r["dense16"], dense)
    assert r["dense16"].size == tiles.size * 1024


def test_s5_raster_layout_against_pixel_coordinates():
    # the C oracle's nest2xyf gives (ix, iy) in the face; inside an NSIDE-256 tile the image position is (ix mod side,
    # iy mod side), x fastest -- independent of raster_offset's bit loop
    rng = np.random.default_rng(12)
    nside, nside_tile = 1 << 17, 1 << 8
    side = nside // nside_tile
    p = rng.integers(0, 12 * nside * nside, 4000)
    off = seg.raster_offset(p & (side * side - 1), side)
    for pi, oi in zip(p.tolist(), off.tolist()):
        _face, ix, iy = oracle.nest2xyf(nside, pi)
        assert oi == (iy % side) * side + (ix % side)
    assert sorted(seg.raster_offset(np.arange(64 * 64), 64).tolist()) == list(range(64 * 64))   # a permutation
    assert seg.raster_offset(np.array([0, 1, 2, 3, 4]), 512).tolist() == [0, 1, 512, 513, 2]
    # through segment_products: same multiset per tile, placed by brute force
    nside, nside_mini, nside_tile = 1 << 10, 1 << 7, 1 << 5
    idx, value, weight = _random_footprint(rng, nside, 5000)
    tiles = np.unique(idx // 1024)
    r = seg.segment_products(idx, value, weight, nside, nside_mini, np.unique(idx // 64), layout_tiles=tiles, nside_tile=nside_tile, raster=True)
    dense = np.zeros(tiles.size * 1024, np.uint16)
    tl = tiles.tolist()
    for pi, b in zip(idx.tolist(), r["seg16"].tolist()):
        _face, ix, iy = oracle.nest2xyf(nside, pi)
        dense[tl.index(pi // 1024) * 1024 + (iy % 32) * 32 + (ix % 32)] = b
    assert np.array_equal(r["dense16"], dense)


def test_empty_and_errors():
    e = np.zeros(0, np.int64)
    r = seg.segment_products(e, np.zeros(0, np.float32), np.zeros(0, np.float32), 1 << 17, 1 << 14, e)
    assert all(r[k].size == 0 for k in ("mini_id", "mini_keep", "mini_weight", "mini_value", "seg16"))
    with pytest.raises(ValueError):
        seg.minipix_of([1], 1 << 10, 1 << 11)
    with pytest.raises(ValueError):
        seg.minipix_of([1], 1 << 10, 48)
