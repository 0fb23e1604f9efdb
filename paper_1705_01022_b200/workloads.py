"""Seeded synthetic workloads shared by the tests, the bench, the oracle side and the CUDA side.

This module holds NONE of the method's arithmetic (no update rule, no RNG of the method, no domain
decomposition): only (a) the parameter sets of the five BASELINE.json configs, (b) the bit layout of
the public `scheme` code and of the canonical packed lattice (both are the boundary's data format,
include/oct.h), and (c) a generator of arbitrary valid slope fields that is unrelated to the dynamics
(used to feed the height-reconstruction and reduction kernels, and to pin the oracle's heights).

The paper uses no dataset: its workloads are square periodic power-of-two lattices started flat and
driven with p=1, q=0, so the configs below *are* the paper's workload shape.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

# ---- public scheme code (include/oct.h): dev | blk<<4 | tcx<<8 | tcy<<12 | log2D<<16 -------------
DEV_DTR, DEV_DT, DEV_DB, DEV_CDB, DEV_DBH = 0, 1, 2, 3, 4
BLK_DB, BLK_DB_DELAYED, BLK_DT, BLK_DTR = 0, 1, 2, 3
INIT_FLAT, INIT_FLAT_SHIFTED, INIT_FROM_DEVICE = 0, 1, 2


def scheme_code(dev: int, blk: int, log2D: int, tcx: int = 1, tcy: int = 1) -> int:
    return dev | (blk << 4) | (tcx << 8) | (tcy << 12) | (log2D << 16)


def scheme_name(code: int) -> str:
    dev, blk = code & 15, (code >> 4) & 15
    return (["DTr", "DT", "DB", "cDB", "DBh"][dev] + ["DB", "DBd", "DT", "DTr"][blk]
            + f",TC={(code >> 8) & 15},{(code >> 12) & 15},D={1 << ((code >> 16) & 31)}")


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    p: float
    q: float
    n_mcs: int
    seeds: tuple
    scheme: int
    note: str


DTRDB = lambda lD: scheme_code(DEV_DTR, BLK_DB, lD)    # noqa: E731  the recommended scheme

# BASELINE.json `configs`, in order.  D per config follows SURVEY.md section 8(a).
CONFIGS = (
    Config("c0_L256", 256, 1.0, 0.0, 100, (1,), DTRDB(6), "64x64 block domains, full oracle run"),
    Config("c1_L1024", 1024, 1.0, 0.0, 2000, tuple(range(1, 9)), DTRDB(7), "all DD schemes vs RS, W2 and C(t,s)"),
    Config("c2_L4096", 4096, 0.9, 0.1, 5000, (7,), DTRDB(7), "mixed deposition/removal (delayed borders)"),
    Config("c3_L65536", 1 << 16, 1.0, 0.0, 10_000, (1,), DTRDB(8), "throughput headline"),
    Config("c4_L131072", 1 << 17, 1.0, 0.0, 10_000, (1,), DTRDB(8), "largest single-GPU lattice, aging run"),
)

# every device-layer scheme the paper defines (Sec. 3) with the block layer of its Fig. 3(b) (DT) and
# with the recommended DB block layer
ALL_SCHEMES = lambda lD: tuple(scheme_code(d, b, lD) for d in (DEV_DTR, DEV_DT, DEV_DB, DEV_CDB)  # noqa: E731
                               for b in (BLK_DB, BLK_DT))


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


def rank_seed(base_seed: int, rank: int) -> int:
    """Replica seeds for `bench.py --gpus N` (replicas only; no data-path collective)."""
    return base_seed + 1_000_003 * rank
