"""Seeded inputs for the segment-product tests: footprint-like pixel lists with values and
weights, and target lists.  No HEALPix arithmetic here: a "footprint" is an ascending list of integers with
gaps, a target list is a random subset of an integer range the caller names.

Draw order (numpy PCG64(seed)): start, hole mask, value, bright mask, bright value, weight-zero mask, weight.
"""
from __future__ import annotations

import numpy as np


def footprint_like(seed, n_universe, n, hole_frac=0.3, start=None, run=4096):
    """n ascending unique int64 in [0, n_universe): runs of consecutive integers `run` long with holes punched at
    rate hole_frac, the way a frame border cuts HEALPix tiles.  Returns idx, value f32 (ADU-like: N(1200, 400),
    1 % bright up to 7e4, which exceeds the binary16 range), weight f32 (10 % zeros, else U(0.5, 1))."""
    rng = np.random.Generator(np.random.PCG64(seed))
    span = int(n / max(1e-3, 1.0 - hole_frac) * 1.5) + 2 * run + 8
    if start is None:
        start = int(rng.integers(0, max(1, n_universe - span)))
    cand = start + np.arange(min(span, n_universe - start), dtype=np.int64)
    keep = rng.random(cand.size) >= hole_frac
    keep[(np.arange(cand.size) // run) % 5 == 3] = False      # whole runs missing: jumps between minipix and tiles
    idx = cand[keep][:n]
    value = rng.normal(1200.0, 400.0, idx.size)
    bright = rng.random(idx.size) < 0.01
    value = np.where(bright, rng.uniform(-100.0, 7.0e4, idx.size), value).astype(np.float32)
    wz = rng.random(idx.size) < 0.1
    weight = np.where(wz, 0.0, rng.uniform(0.5, 1.0, idx.size)).astype(np.float32)
    return idx, value, weight


def target_list(seed, lo, hi, frac, n_foreign=5):
    """Random ids from [lo, hi) (a fraction frac of them), a few from outside, some duplicated, shuffled."""
    rng = np.random.Generator(np.random.PCG64(seed))
    m = int(hi - lo)
    pick = lo + np.flatnonzero(rng.random(m) < frac).astype(np.int64) if m > 0 else np.zeros(0, np.int64)
    foreign = np.concatenate([lo - 1 - rng.integers(0, 1000, n_foreign), hi + rng.integers(0, 1000, n_foreign)]).astype(np.int64)
    foreign = foreign[foreign >= 0]
    dup = pick[: min(7, pick.size)]
    t = np.concatenate([pick, foreign, dup])
    rng.shuffle(t)
    return t
