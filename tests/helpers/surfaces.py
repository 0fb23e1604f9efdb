"""Seeded synthetic surfaces for the tests (both sides): the canonical packed format written out from a height
array, and a generator of valid periodic surfaces that is unrelated to the dynamics.  Holds none of the method's
arithmetic (no update rule, no RNG of the method, no domain decomposition); it pins the oracle's packing and
heights (tests/test_oracle_rule.py) and feeds the height-reconstruction / reduction kernels rough inputs.
"""
from __future__ import annotations

import numpy as np


# ---- canonical packed format (include/oct.h; "each 32-bit word encodes 4x4 sites") ----
def pack_slopes(sx: np.ndarray, sy: np.ndarray) -> np.ndarray:
    """sx, sy: (L, L) arrays indexed [y, x] of 0/1 bits (1 <=> slope +1 towards the site from its
    west / south neighbour).  Returns (L/4, L/4) uint32 words: site (4wx+i, 4wy+j) has sigma_x at bit
    2(4j+i) and sigma_y at bit 2(4j+i)+1 of word [wy, wx]."""
    L = sx.shape[0]
    assert sx.shape == (L, L) and sy.shape == (L, L) and L % 4 == 0
    n = L // 4
    out = np.zeros((n, n), dtype=np.uint32)
    for j in range(4):
        for i in range(4):
            b = 2 * (4 * j + i)
            out |= (sx[j::4, i::4].astype(np.uint32) & 1) << np.uint32(b)
            out |= (sy[j::4, i::4].astype(np.uint32) & 1) << np.uint32(b + 1)
    return out


def pack_heights(h: np.ndarray) -> np.ndarray:
    """Canonical words of a periodic height field h[y, x] whose neighbours differ by exactly 1."""
    dx = h - np.roll(h, 1, axis=1)
    dy = h - np.roll(h, 1, axis=0)
    assert (np.abs(dx) == 1).all() and (np.abs(dy) == 1).all(), "not a valid octahedron surface"
    return pack_slopes((dx == 1), (dy == 1))


def _balanced_walk(rng: np.random.Generator, L: int) -> np.ndarray:
    steps = np.array([1] * (L // 2) + [-1] * (L // 2), dtype=np.int32)
    rng.shuffle(steps)
    return np.cumsum(steps).astype(np.int32) - steps[0]        # w[0] = 0, |w[i+1]-w[i]| = 1, periodic


def separable_surface(L: int, seed: int, offset: int = 0) -> np.ndarray:
    """A valid periodic surface unrelated to the dynamics: h[y, x] = a[x] + b[y] + offset with a, b
    closed +-1 walks.  h[0, 0] = offset.  Rough (|h| ~ sqrt(L)), so it exercises carries and signs."""
    rng = np.random.default_rng(seed)
    a, b = _balanced_walk(rng, L), _balanced_walk(rng, L)
    return (a[None, :] + b[:, None] + offset).astype(np.int32)
