"""Pins P1-P4 for the oracle's HEALPix layer (O2, O3, O3b): checked against what the HEALPix
definition fixes, not against the oracle itself (BASELINE.json north_star)."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _centres(nside):
    n = 12 * nside * nside
    th = np.empty(n)
    ph = np.empty(n)
    for p in range(n):
        th[p], ph[p] = oracle.pix2ang(nside, p)
    return th, ph


def test_p1_nside1_base_pixel_centres():
    rows = [l.split() for l in open(os.path.join(GOLD, "nside1_centres.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 12
    for r in rows:
        p = int(r[0])
        z = float(Fraction(int(r[1]), int(r[2])))
        phi = math.pi * float(Fraction(int(r[3]), int(r[4])))
        th, ph = oracle.pix2ang(1, p)
        assert abs(math.cos(th) - z) < 1e-15
        assert abs(ph - phi) < 1e-15


def test_paper_facts():
    facts = {}
    for l in open(os.path.join(GOLD, "paper_facts.txt")):
        if l.strip() and l[0] != "#":
            k, v = l.split()[:2]
            facts[k] = float(v)
    assert 12 * 256 ** 2 == facts["n_tiles_nside256"]
    side = math.degrees(math.sqrt(4 * math.pi / (12 * 256 ** 2))) * 60
    assert abs(side - facts["tile_side_arcmin"]) < 0.05
    assert facts["minipix_nside"] == 256 * 64
    assert round(9576 * 6388 / 1e6) == facts["frame_mpix"]
    assert round(9576 * 6388 * 2 / 1e6) == facts["frame_mbytes"]
    # fraction of equal-area tiles whose centre lies north of dec0: (1 - sin dec0)/2 = 0.586 -> dec0 ~ -9.9 deg
    n = 12 * 256 * 256
    rng = np.random.default_rng(0)
    ps = rng.integers(0, n, 4000)
    z = np.array([math.cos(oracle.pix2ang(256, int(p))[0]) for p in ps])
    dec0 = math.asin(1 - 2 * facts["north_fraction"])
    assert abs((z > math.sin(dec0)).mean() - facts["north_fraction"]) < 0.03


def _ring_centres(N):
    """Textbook RING-scheme closed form (Gorski et al. 2005): ring i has z_i and equally spaced phi_j."""
    out = []
    for i in range(1, N):  # north cap
        z = 1 - i * i / (3.0 * N * N)
        for j in range(1, 4 * i + 1):
            out.append((z, math.pi / (2 * i) * (j - 0.5)))
    for i in range(N, 3 * N + 1):  # belt
        z = 4.0 / 3.0 - 2.0 * i / (3.0 * N)
        s = (i - N + 1) % 2
        for j in range(1, 4 * N + 1):
            out.append((z, math.pi / (2 * N) * (j - s / 2.0)))
    for i in range(N - 1, 0, -1):  # south cap
        z = -(1 - i * i / (3.0 * N * N))
        for j in range(1, 4 * i + 1):
            out.append((z, math.pi / (2 * i) * (j - 0.5)))
    return out


@pytest.mark.parametrize("nside", [1, 2, 4, 8, 16, 32, 64])
def test_p2_nested_centres_equal_ring_centres(nside):
    ring = _ring_centres(nside)
    assert len(ring) == 12 * nside * nside
    th, ph = _centres(nside)
    a = np.array(sorted((round(z, 11), round(p % (2 * math.pi), 11)) for z, p in ring))
    b = np.array(sorted((round(float(math.cos(t)), 11), round(float(p), 11)) for t, p in zip(th, ph)))
    assert np.abs(a - b).max() < 2e-11


@pytest.mark.parametrize("nside", [1, 2, 4, 16, 64])
def test_p3_roundtrip_all_pixels(nside):
    for p in range(12 * nside * nside):
        th, ph = oracle.pix2ang(nside, p)
        assert oracle.ang2pix(nside, th, ph) == p


@pytest.mark.parametrize("k", [10, 17, 18, 29])
def test_p3_roundtrip_random_high_nside(k):
    nside = 1 << k
    rng = np.random.default_rng(k)
    ps = rng.integers(0, 12 * nside * nside, 60000, dtype=np.int64)
    for p in ps:
        th, ph = oracle.pix2ang(nside, int(p))
        assert oracle.ang2pix(nside, th, ph) == int(p)


def test_p3_xyf_roundtrip_and_bit_layout():
    nside = 1 << 17
    # ix occupies the even bits, iy the odd bits, face the top bits
    assert oracle.xyf2nest(nside, 0, 1, 0) == 1
    assert oracle.xyf2nest(nside, 0, 0, 1) == 2
    assert oracle.xyf2nest(nside, 0, 2, 0) == 4
    assert oracle.xyf2nest(nside, 5, 0, 0) == 5 * nside * nside
    rng = np.random.default_rng(1)
    for _ in range(2000):
        f, ix, iy = int(rng.integers(12)), int(rng.integers(nside)), int(rng.integers(nside))
        assert oracle.nest2xyf(nside, oracle.xyf2nest(nside, f, ix, iy)) == (f, ix, iy)


def test_p4_hierarchy_equal_area():
    """Each coarse pixel receives exactly 256 fine centres (nested hierarchy) => 12 nside^2 pixels of
    equal area 4 pi / (12 nside^2)."""
    N = 4
    counts = np.zeros(12 * N * N, dtype=np.int64)
    for q in range(12 * (16 * N) ** 2):
        th, ph = oracle.pix2ang(16 * N, q)
        c = oracle.ang2pix(N, th, ph)
        assert c == q >> 8
        counts[c] += 1
    assert np.all(counts == 256)


def test_p4_ang2pix_equal_area_monte_carlo():
    """Independent of pix2ang: uniform points on the sphere land uniformly in the 192 nside=4 pixels."""
    rng = np.random.default_rng(7)
    n = 192 * 1500
    z = rng.uniform(-1, 1, n)
    phi = rng.uniform(0, 2 * math.pi, n)
    th = np.arccos(z)
    counts = np.zeros(192)
    for t, p in zip(th, phi):
        counts[oracle.ang2pix(4, float(t), float(p))] += 1
    chi2 = ((counts - 1500) ** 2 / 1500).sum()
    assert chi2 < 191 + 5 * math.sqrt(2 * 191)  # 5 sigma


@pytest.mark.parametrize("nside", [8, 32])
def test_p4_symmetries(nside):
    th, ph = _centres(nside)
    v = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)], 1)
    assert np.abs(v.sum(0)).max() < 1e-9  # centroid of all centres is the origin
    # z-antisymmetry: the multiset of z is symmetric, and each (z, phi) has a partner (-z, phi)
    a = sorted((round(float(math.cos(t)), 11), round(float(p), 11)) for t, p in zip(th, ph))
    b = sorted((round(float(-math.cos(t)), 11), round(float(p), 11)) for t, p in zip(th, ph))
    assert np.abs(np.array(a) - np.array(b)).max() < 2e-11
    # four-fold symmetry in phi
    c = sorted((round(float(math.cos(t)), 11), round(float((p + math.pi / 2) % (2 * math.pi)), 11) % round(2 * math.pi, 11))
               for t, p in zip(th, ph))
    assert np.abs(np.array(a) - np.array(c)).max() < 2e-11


def test_pixel_neighbour_spacing():
    """Adjacent (ix+1) centres at nside 2^17 are ~ one pixel side apart: sqrt(4 pi/(12 nside^2))."""
    nside = 1 << 17
    side = math.sqrt(4 * math.pi / (12.0 * nside * nside))
    rng = np.random.default_rng(3)
    for _ in range(300):
        f, ix, iy = int(rng.integers(12)), int(rng.integers(nside - 1)), int(rng.integers(nside - 1))
        t0, p0 = oracle.pix2ang(nside, oracle.xyf2nest(nside, f, ix, iy))
        t1, p1 = oracle.pix2ang(nside, oracle.xyf2nest(nside, f, ix + 1, iy))
        d = math.hypot(t1 - t0, math.sin(t0) * ((p1 - p0 + math.pi) % (2 * math.pi) - math.pi))
        assert 0.5 * side < d < 1.6 * side  # pixels are sheared near the poles
