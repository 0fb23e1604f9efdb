"""Host-side logic of `bench.py --gpus N`: N independent replicas, one process per GPU.

The path does not shard (BASELINE.json north_star: one GPU, no collectives; the paper's statistics come
from hundreds of independent runs): every rank owns a whole lattice with its own seed,
there is no data-path collective, and the only communication is the bench's own barrier and the
max-over-ranks of the timings.  This module holds that logic so it can be tested on CPU with `gloo`.
"""
from __future__ import annotations

from . import workloads as wl


def replica_seed(base_seed: int, rank: int) -> int:
    return wl.rank_seed(base_seed, rank)


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise maximum of a list of floats over all ranks (identity when not distributed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def gather_ints(value: int, dist=None, device="cpu"):
    """All ranks' integer `value`, in rank order."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [int(value)]
    import torch
    mine = torch.tensor([int(value)], dtype=torch.int64, device=device)
    out = [torch.zeros_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine)
    return [int(o.cpu()[0]) for o in out]


def aggregate_throughput(units_per_rank_per_step: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job units per second: every rank processed the same number of units (weak scaling) and the
    job took as long as its slowest rank."""
    return world * steps * units_per_rank_per_step / (max_ms * 1e-3)
