"""N > 1 path of bench.py on CPU: world_size-2 `gloo` run of the replica bookkeeping (seeds, barrier,
max-over-ranks timing, aggregate throughput).  The replicas exchange no lattice data by design."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist          # noqa: E402
import torch.multiprocessing as mp        # noqa: E402

from paper_1705_01022_b200 import replicas  # noqa: E402


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = replicas.replica_seed(1, rank)
        seeds = replicas.gather_ints(seed, dist)
        dist.barrier()
        # rank r pretends to have taken (10 + 5 r) ms for the step and (7 - r) ms for the sweeps
        total_ms, sweep_ms = replicas.max_over_ranks([10.0 + 5.0 * rank, 7.0 - rank], dist)
        value = replicas.aggregate_throughput(units_per_rank_per_step=1000, steps=4, world=world, max_ms=total_ms)
        q.put((rank, seed, seeds, total_ms, sweep_ms, value))
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, all0, t0, w0, v0), (r1, s1, all1, t1, w1, v1) = out
    assert (r0, r1) == (0, 1) and s0 != s1 and all0 == all1 == [s0, s1]      # independent seeds, same view on both ranks
    assert t0 == t1 == 15.0 and w0 == w1 == 7.0                               # max over ranks, per quantity
    assert v0 == v1 == pytest.approx(2 * 4 * 1000 / 15e-3)                    # whole-job units / slowest rank


def test_single_process_is_the_identity():
    assert replicas.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
    assert replicas.gather_ints(7) == [7]
    assert replicas.replica_seed(5, 0) == 5 and replicas.replica_seed(5, 1) != replicas.replica_seed(5, 2)
