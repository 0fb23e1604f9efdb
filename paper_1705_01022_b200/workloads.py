"""Seeded synthetic workloads shared by the tests, the bench, the oracle side and the CUDA side.

This module holds NONE of the method's arithmetic (no update rule, no RNG of the method, no domain
decomposition): only (a) the parameter sets of the five BASELINE.json configs and (b) the bit layout of
the public `scheme` code (the boundary's data format, include/oct.h).  The generator of arbitrary valid
surfaces that feeds the reconstruction / reduction kernels and pins the oracle's heights is test
infrastructure and lives in tests/helpers/surfaces.py.

The paper uses no dataset: its workloads are square periodic power-of-two lattices started flat and
driven with p=1, q=0, so the configs below *are* the paper's workload shape.
"""
from __future__ import annotations

from dataclasses import dataclass

# ---- public scheme code (include/oct.h): dev | blk<<4 | tcx<<8 | tcy<<12 | log2D<<16 | ka<<21 | w<<23 ----
DEV_DTR, DEV_DT, DEV_DB, DEV_CDB, DEV_DBH = 0, 1, 2, 3, 4
BLK_DB, BLK_DB_DELAYED, BLK_DT, BLK_DTR = 0, 1, 2, 3
INIT_FLAT, INIT_FLAT_SHIFTED, INIT_FROM_DEVICE = 0, 1, 2


def scheme_code(dev: int, blk: int, log2D: int, tcx: int = 1, tcy: int = 1, ka: int = 0, w: int = 0) -> int:
    """ka: t_async = 2^-ka MCS; w: explicit dead-border width, 0 = the scheme's own (DB / cDB only)."""
    return dev | (blk << 4) | (tcx << 8) | (tcy << 12) | (log2D << 16) | (ka << 21) | (w << 23)


def scheme_name(code: int) -> str:
    dev, blk = code & 15, (code >> 4) & 15
    ka, w = (code >> 21) & 3, (code >> 23) & 7
    return (["DTr", "DT", "DB", "cDB", "DBh"][dev] + ["DB", "DBd", "DT", "DTr"][blk]
            + f",TC={(code >> 8) & 15},{(code >> 12) & 15},D={1 << ((code >> 16) & 31)}"
            + (f",tasync=1/{1 << ka}" if ka else "") + (f",w={w}" if w else ""))


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


def rank_seed(base_seed: int, rank: int) -> int:
    """Replica seeds for `bench.py --gpus N` (replicas only; no data-path collective)."""
    return base_seed + 1_000_003 * rank
