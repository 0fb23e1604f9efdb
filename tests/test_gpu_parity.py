"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

Everything is integer work, so the bar is exact equality of lattice words, heights, counters and sums
for the same (L, seed, init, scheme, p, q).  Sizes span one to many device-layer domains, several
worker-group shapes, ragged word windows (random origins), wrap-around and the degenerate L = 2D.
"""
import numpy as np
import pytest

import oracle
from oracle import Oracle
from helpers import surfaces as sf
from paper_1705_01022_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def gpu_run(L, seed, code, n, p, q, init=wl.INIT_FLAT, chunks=None, kernel=binding.OCT_KERNEL_AUTO):
    sim = binding.Sim(L, seed, init)
    sim.oct_set_option(binding.OCT_OPT_KERNEL, kernel)
    for c in (chunks or [n]):
        sim.oct_sweep(c, p, q, code)
    return sim


def compare_state(sim, orc, check_heights=True):
    words = sim.oct_export()
    assert (words == orc.lattice).all(), f"{(words != orc.lattice).sum()} of {words.size} words differ"
    h00, net = sim.oct_counters()
    assert (h00, net) == (orc.h00, orc.net)
    assert sim.oct_mcs() == orc.t
    S = sim.oct_width2().cpu().numpy()
    assert tuple(int(v) for v in S) == orc.sums()
    if check_heights:
        h = sim.oct_heights().cpu().numpy()
        assert (h == orc.heights()).all()


SMALL = [
    # (L, code, p, q, n_mcs)
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 1.0, 0.0, 20),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 0.0, 1.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 0.9, 0.1, 12),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB_DELAYED, 6), 1.0, 0.0, 8),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6), 1.0, 0.0, 12),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6), 0.7, 0.3, 8),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 6), 1.0, 0.0, 8),              # "DTrDTr"
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 7, 2, 1), 0.7, 0.3, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 8), 1.0, 0.0, 3),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DTR, 6), 0.6, 0.4, 4),
    (256, wl.scheme_code(wl.DEV_DT, wl.BLK_DB, 6), 1.0, 0.0, 8),
    (256, wl.scheme_code(wl.DEV_DT, wl.BLK_DT, 6), 1.0, 0.0, 8),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6), 1.0, 0.0, 8),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DT, 6), 0.6, 0.4, 8),
    (256, wl.scheme_code(wl.DEV_DBH, wl.BLK_DB, 6), 1.0, 0.0, 8),               # DB with t_async = 1/2
    (256, wl.scheme_code(wl.DEV_DBH, wl.BLK_DT, 6), 0.7, 0.3, 4),
    (512, wl.scheme_code(wl.DEV_DBH, wl.BLK_DB, 8), 0.9, 0.1, 3),
    (256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DB, 6), 1.0, 0.0, 8),
    (256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DT, 6), 1.0, 0.0, 8),
    (64, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5), 1.0, 0.0, 16),               # L = 2D: a single tile
    (64, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6), 1.0, 0.0, 12),                # L = D: a single dead-border tile
    (64, wl.scheme_code(wl.DEV_CDB, wl.BLK_DT, 6), 0.7, 0.3, 8),
    (32, wl.scheme_code(wl.DEV_DBH, wl.BLK_DB, 5), 0.9, 0.1, 12),
    (128, wl.scheme_code(wl.DEV_CDB, wl.BLK_DB, 7), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 8), 0.8, 0.2, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 2, 2), 0.9, 0.1, 5),         # two domains per warp, delayed borders
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6, 2, 2), 0.6, 0.4, 5),
    (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 2, 2), 1.0, 0.0, 6),          # ... of which one has no domain (4 tiles, odd split)
    (64, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 5), 0.5, 0.5, 10),               # D = 32 TC=1,1: half-warp groups, one tile
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 2, 0), 1.0, 0.0, 8),    # t_async = 1/4 MCS
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 0, 1), 1.0, 0.0, 10),   # border width 1 with a FREE origin: shared words
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 1, 1), 0.7, 0.3, 8),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DT, 6, 1, 1, 2, 3), 0.6, 0.4, 6),
    (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 5, 1, 1, 2, 2), 0.9, 0.1, 8),
    (256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DB, 6, 1, 1, 2, 3), 1.0, 0.0, 6),
    (512, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 7, 1, 1, 1, 1), 1.0, 0.0, 4),
    (512, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 8, 1, 1, 2, 1), 0.8, 0.2, 3),    # D = 256: 16-bit coordinate fields, bit-wise write-back
    (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 2, 2, 1, 1), 1.0, 0.0, 6),    # two domains per warp
    (64, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 2, 1), 0.7, 0.3, 10),    # L = D, width 1: the tile is its own neighbour
    (64, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 5), 0.5, 0.5, 16),
    (128, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5, 0, 0), 1.0, 0.0, 8),
    (128, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5, 2, 2), 0.8, 0.2, 8),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 0, 0), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 2, 2), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6, 2, 1), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 3, 1), 0.9, 0.1, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6, 1, 3), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7), 1.0, 0.0, 8),               # one warp, 8 cells per lane
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7), 0.9, 0.1, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 7), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 0, 0), 1.0, 0.0, 4),         # 4 warps per domain
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 2, 2), 0.9, 0.1, 4),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 3, 2), 1.0, 0.0, 3),         # Fig. 4 cell shapes at D = 128
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 7, 4, 1), 1.0, 0.0, 3),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 4, 1), 0.8, 0.2, 2),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8), 1.0, 0.0, 6),               # D = 256: one 512-thread CTA per domain, two-byte entries, __syncthreads
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8), 0.9, 0.1, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 8), 1.0, 0.0, 4),
    (512, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 8), 1.0, 0.0, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8, 2, 2), 1.0, 0.0, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8, 3, 2), 0.9, 0.1, 4),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 8, 4, 1), 1.0, 0.0, 4),
    # the remaining cell shapes of the Fig. 4 caption on the link-entry kernel: TC=3,1 / 1,3 at D = 64 (16 cells:
    # half-warp groups) and D = 128 (64 cells), TC=3,2 / 4,1 at D = 256 (128 cells); every block layer, dead borders too
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 3, 1), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB_DELAYED, 6, 1, 3), 1.0, 0.0, 4),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 1, 3), 0.9, 0.1, 5),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 6, 3, 1), 0.7, 0.3, 4),
    (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 3, 1, 1), 1.0, 0.0, 6),
    (256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DT, 6, 3, 1), 0.6, 0.4, 4),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 3, 1), 1.0, 0.0, 4),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 1, 3), 0.8, 0.2, 3),
    (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 7, 3, 1), 1.0, 0.0, 3),
    (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 7, 1, 3, 2, 1), 0.7, 0.3, 3),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8, 3, 2), 1.0, 0.0, 3),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8, 4, 1), 0.9, 0.1, 3),
    (512, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 8, 4, 1, 1, 1), 1.0, 0.0, 3),
    (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 8, 3, 2), 0.6, 0.4, 2),
]


KERNELS = {"auto": binding.OCT_KERNEL_AUTO, "bitpacked": binding.OCT_KERNEL_BITPACKED, "linksB": binding.OCT_KERNEL_LINKS_B}


@pytest.mark.parametrize("L,code,p,q,n", SMALL, ids=[f"L{c[0]}-{wl.scheme_name(c[1])}-p{c[2]}q{c[3]}" for c in SMALL])
def test_sweep_bit_exact(L, code, p, q, n):
    """Every kernel the library can pick for a scheme (link-entry, its alternative work split, bit-packed)
    gives the oracle's lattice, counters, sums and heights."""
    seed = 1000 + L + (code & 0xFFFF)
    orc = Oracle(L, seed)
    orc.sweep(n, p, q, code)
    for name, k in KERNELS.items():
        sim = gpu_run(L, seed, code, n, p, q, kernel=k)
        compare_state(sim, orc, check_heights=(name == "auto"))
        sim.close()
    orc.close()


SEEDS64 = (0x9E3779B97F4A7C15, (7 << 32) | 1, 1 << 32)


@pytest.mark.parametrize("seed", SEEDS64, ids=[hex(s) for s in SEEDS64])
def test_seeds_with_a_high_half_reach_every_kernel_family(seed):
    """The Philox key is the 64-bit seed as (low word, high word) (R19).  Every other case in this file has a seed
    below 2^32, i.e. a zero second key word: here the high half is live in each kernel family -- four-byte link
    entries, two-byte entries (TC=2,2 at D = 64, D = 256), the alternative work split, the bit-packed kernel, a
    dead-border layer, delayed borders, the DT block layer."""
    cases = [(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 1.0, 0.0, 4),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 0.9, 0.1, 4),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 2, 2), 1.0, 0.0, 3),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 7), 0.7, 0.3, 3),
             (256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 1, 1), 1.0, 0.0, 3),
             (512, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 8), 1.0, 0.0, 2)]
    for L, code, p, q, n in cases:
        orc = Oracle(L, seed)
        orc.sweep(n, p, q, code)
        low = Oracle(L, seed & 0xFFFFFFFF)
        low.sweep(n, p, q, code)
        assert (low.lattice != orc.lattice).any(), "the high half of the seed does not reach the oracle's streams"
        low.close()
        for name, k in KERNELS.items():
            sim = gpu_run(L, seed, code, n, p, q, kernel=k)
            compare_state(sim, orc, check_heights=False)
            sim.close()
        orc.close()


def test_batch_members_that_differ_only_in_the_high_half_of_the_seed():
    """oct_sweep_batch builds each member's round keys in registers from (seed_lo, seed_hi): members with one low word
    and different high words must each follow their own oracle run."""
    L, n = 256, 3
    for code, p, q in ((wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 1.0, 0.0), (wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 2, 2), 0.8, 0.2),
                       (wl.scheme_code(wl.DEV_DB, wl.BLK_DT, 6), 0.6, 0.4), (wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7), 1.0, 0.0)):
        seeds = [5, (1 << 32) | 5, (0xDEADBEEF << 32) | 5, (1 << 63) | 5]
        sims = [binding.Sim(L, sd) for sd in seeds]
        binding.oct_sweep_batch(sims, n, p, q, code)
        words = []
        for sim, sd in zip(sims, seeds):
            orc = Oracle(L, sd)
            orc.sweep(n, p, q, code)
            compare_state(sim, orc, check_heights=False)
            words.append(orc.lattice.copy())
            orc.close()
            sim.close()
        for i in range(len(words)):
            for j in range(i):
                assert (words[i] != words[j]).any()


def test_a_second_device_in_the_same_process():
    """One process may drive several GPUs (replicas are this path's only multi-GPU mode): the > 48 KiB shared-memory
    opt-in is per device, so a shape that needs it (D = 128: 70 KiB) must also launch on the second device used."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    L, code, n = 256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7), 3
    orc = Oracle(L, 21)
    orc.sweep(n, 1.0, 0.0, code)
    try:
        for dev in ("cuda:0", "cuda:1", "cuda:0"):
            sim = binding.Sim(L, 21, device=dev)          # makes `dev` current
            sim.oct_sweep(n, 1.0, 0.0, code)
            compare_state(sim, orc, check_heights=False)
            sim.close()
    finally:
        torch.cuda.set_device(0)
    orc.close()


def test_origin_site_height_is_tracked_when_it_is_updated():
    """The tracked anchor h(0,0) (R20) moves only when site (0,0) itself is updated: long enough runs on a
    small lattice that it moves many times, both directions, all kernels."""
    L = 64
    for code, p, q in ((wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5, 0, 0), 1.0, 0.0), (wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5, 0, 0), 0.0, 1.0),
                       (wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5, 0, 0), 0.6, 0.4), (wl.scheme_code(wl.DEV_DT, wl.BLK_DT, 5, 1, 1), 0.7, 0.2)):
        orc = Oracle(L, 77); orc.sweep(60, p, q, code)
        assert orc.h00 != 0
        for k in KERNELS.values():
            sim = gpu_run(L, 77, code, 60, p, q, kernel=k)
            compare_state(sim, orc, check_heights=False)
            sim.close()
        orc.close()


def test_config0_L256_100mcs_per_mcs_sums():
    """BASELINE config 1: L=256, D=64, p=1,q=0, 100 MCS, seed 1: lattice, heights and W^2(t) per MCS."""
    cfg = wl.CONFIGS[0]
    orc = Oracle(cfg.L, cfg.seeds[0])
    sim = binding.Sim(cfg.L, cfg.seeds[0])
    for t in range(cfg.n_mcs):
        orc.sweep(1, cfg.p, cfg.q, cfg.scheme)
        sim.oct_sweep(1, cfg.p, cfg.q, cfg.scheme)
        S = tuple(int(v) for v in sim.oct_width2().cpu().numpy())
        assert S == orc.sums(), t
        assert binding.oct_w2_from_sums(cfg.L, S[0], S[1]) == pytest.approx(float(orc.w2()), rel=1e-14)
    compare_state(sim, orc)
    sim.close(); orc.close()


def test_split_invariance_and_resume():
    L, code = 256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)
    a = gpu_run(L, 5, code, 9, 1.0, 0.0)
    b = gpu_run(L, 5, code, 9, 1.0, 0.0, chunks=[2, 0, 3, 4])
    assert (a.oct_export() == b.oct_export()).all() and a.oct_counters() == b.oct_counters()
    # resume from an exported lattice on a fresh handle
    words = a.oct_export()
    h00, net = a.oct_counters()
    c = binding.Sim(L, 5, wl.INIT_FROM_DEVICE, lattice=torch.from_numpy(words.view(np.int32).reshape(-1)).cuda())
    c.oct_set_state(9, h00, net)
    a.oct_sweep(3, 1.0, 0.0, code); c.oct_sweep(3, 1.0, 0.0, code)
    assert (a.oct_export() == c.oct_export()).all() and a.oct_counters() == c.oct_counters()
    orc = Oracle(L, 5); orc.sweep(12, 1.0, 0.0, code)
    compare_state(c, orc)
    for s in (a, b, c):
        s.close()
    orc.close()


def test_flat_shifted_symmetry_on_gpu():
    L, code = 256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)
    a = gpu_run(L, 3, code, 5, 0.8, 0.3, init=wl.INIT_FLAT)
    b = gpu_run(L, 3, code, 5, 0.3, 0.8, init=wl.INIT_FLAT_SHIFTED)
    assert (a.oct_export() == ~b.oct_export()).all()
    ha, na = a.oct_counters(); hb, nb = b.oct_counters()
    assert (ha, na) == (-hb, -nb)
    orc = Oracle(L, 3, init=1); orc.sweep(5, 0.3, 0.8, code)
    compare_state(b, orc)
    a.close(); b.close(); orc.close()


@pytest.mark.parametrize("L,seed,off", [(16, 1, 0), (32, 9, 2), (64, 2, -7), (128, 5, 3), (256, 3, 1000), (1024, 4, -123456),
                                        (2048, 6, 77), (4096, 7, -40000)])
def test_heights_and_sums_on_synthetic_surfaces(L, seed, off):
    """Reconstruction / reduction kernels on surfaces unrelated to the dynamics (rough, ragged L)."""
    h = sf.separable_surface(L, seed, off)
    words = sf.pack_heights(h)
    sim = binding.Sim(L, 0, wl.INIT_FROM_DEVICE, lattice=torch.from_numpy(words.view(np.int32).reshape(-1)).cuda())
    sim.oct_set_state(0, off, 17)
    orc = Oracle(L, 0); orc.set_lattice(words, h00=off, net=17)
    assert (sim.oct_heights().cpu().numpy() == h).all()
    assert tuple(int(v) for v in sim.oct_width2().cpu().numpy()) == orc.sums()
    # autocorrelation against a second, different surface
    h2 = sf.separable_surface(L, seed + 100, off - 5)
    snap = torch.from_numpy(sf.pack_heights(h2).view(np.int32).reshape(-1)).cuda()
    anchor = torch.tensor([off - 5, 3], dtype=torch.int64, device="cuda")
    got = tuple(int(v) for v in sim.oct_autocorr(snap, anchor).cpu().numpy())
    orc2 = Oracle(L, 0); orc2.set_lattice(sf.pack_heights(h2), h00=off - 5, net=3)
    assert got == orc.autocorr_sums(orc2)
    # slope autocorrelation against the same second surface, and C_s(s,s) = 1/4
    cs = tuple(int(v) for v in sim.oct_slope_autocorr(snap).cpu().numpy())
    assert cs == orc.slope_autocorr_sums(orc2)
    own = tuple(int(v) for v in sim.oct_slope_autocorr(sim.lattice).cpu().numpy())
    assert own == (L * L // 2,) * 6
    assert binding.oct_cs_from_sums(2 * L * L, own[0] + own[1], own[2] + own[3], own[4] + own[5]) == 0.25
    assert binding.oct_cs_from_sums(2 * L * L, cs[0] + cs[1], cs[2] + cs[3], cs[4] + cs[5]) == pytest.approx(float(orc.c_s(orc2)), rel=1e-12, abs=1e-15)
    sim.close(); orc.close(); orc2.close()


def test_aging_snapshot_and_autocorrelation():
    L, code = 256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)
    orc = Oracle(L, 8); sim = binding.Sim(L, 8)
    orc.sweep(10, 1.0, 0.0, code); sim.oct_sweep(10, 1.0, 0.0, code)
    osnap = orc.clone()
    snap, anchor = sim.oct_snapshot()
    # C_h(s,s) sums reproduce the W^2 sums
    S = [int(v) for v in sim.oct_width2().cpu().numpy()]
    A = [int(v) for v in sim.oct_autocorr(snap, anchor).cpu().numpy()]
    assert A[0] == A[1] == S[0] and A[2] == S[1] and A[3] == A[4] == S[2]
    for n in (5, 15):
        orc.sweep(n, 1.0, 0.0, code); sim.oct_sweep(n, 1.0, 0.0, code)
        A = tuple(int(v) for v in sim.oct_autocorr(snap, anchor).cpu().numpy())
        assert A == orc.autocorr_sums(osnap)
        assert tuple(int(v) for v in sim.oct_slope_autocorr(snap).cpu().numpy()) == orc.slope_autocorr_sums(osnap)
        assert binding.oct_c_from_sums(L, A[0], A[1], A[2]) == pytest.approx(float(orc.c_h(osnap)), rel=1e-13)
    sim.close(); orc.close(); osnap.close()


def test_config1_shape_all_schemes_L1024_prefix():
    """BASELINE config 2 (L=1024, D=128, every device-layer scheme): first MCS bit-exact per scheme."""
    L = 1024
    for code in wl.ALL_SCHEMES(7):
        orc = Oracle(L, 2); sim = binding.Sim(L, 2)
        orc.sweep(3, 1.0, 0.0, code); sim.oct_sweep(3, 1.0, 0.0, code)
        compare_state(sim, orc, check_heights=False)
        sim.close(); orc.close()


def test_config2_shape_mixed_rates_L4096_prefix():
    """BASELINE config 3 (L=4096, p=0.9, q=0.1, seed 7, D=128, delayed borders): first 2 MCS."""
    cfg = wl.CONFIGS[2]
    orc = Oracle(cfg.L, cfg.seeds[0]); sim = binding.Sim(cfg.L, cfg.seeds[0])
    orc.sweep(2, cfg.p, cfg.q, cfg.scheme); sim.oct_sweep(2, cfg.p, cfg.q, cfg.scheme)
    compare_state(sim, orc, check_heights=False)
    sim.close(); orc.close()


def test_degenerate_calls_change_nothing():
    """p = q = 0 (no update can be accepted) and n_mcs = 0 leave the lattice and the counters alone; the clock
    advances only by the sweeps actually run.  Every kernel."""
    for k in KERNELS.values():
        for code in (wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6), wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6)):
            sim = binding.Sim(256, 4)
            sim.oct_set_option(binding.OCT_OPT_KERNEL, k)
            sim.oct_sweep(3, 1.0, 0.0, code)
            before, cnt = sim.oct_export().copy(), sim.oct_counters()
            sim.oct_sweep(0, 1.0, 0.0, code)
            assert sim.oct_mcs() == 3
            sim.oct_sweep(2, 0.0, 0.0, code)
            assert sim.oct_mcs() == 5 and (sim.oct_export() == before).all() and sim.oct_counters() == cnt
            sim.close()


def test_invalid_calls_are_rejected_without_side_effects():
    sim = binding.Sim(256, 1)
    before = sim.oct_export().copy()
    for args in ((1, 1.5, 0.0, wl.scheme_code(0, 0, 6)), (1, 1.0, -0.1, wl.scheme_code(0, 0, 6)),
                 (1, 1.0, 0.0, wl.scheme_code(0, 0, 8)), (1, 1.0, 0.0, wl.scheme_code(0, 2, 6, 0, 0)),
                 (1 << 33, 1.0, 0.0, wl.scheme_code(0, 0, 6))):
        with pytest.raises(binding.OctError) as e:
            sim.oct_sweep(*args)
        assert e.value.code == binding.OCT_EINVAL
    assert (sim.oct_export() == before).all() and sim.oct_mcs() == 0
    sim.close()


def test_batch_members_equal_their_single_runs_and_the_oracle():
    """oct_sweep_batch (many lattices of one size per launch, PAPER.md:200/:232 ensembles): every member ends bit-identical
    to the oracle run with that member's seed -- also with unequal clocks, for a dead-border layer, for two domains per
    warp, and for a shape that has no batch kernel (members run one after the other)."""
    cases = [(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 1.0, 0.0, 5, 5),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6), 0.8, 0.2, 3, 3),
             (128, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 5), 0.7, 0.3, 3, 260),     # more members than one launch holds (256)
             (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6), 1.0, 0.0, 4, 3),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 2, 2), 1.0, 0.0, 3, 4),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 3, 1), 0.9, 0.1, 3, 5),
             (128, wl.scheme_code(wl.DEV_DB, wl.BLK_DT, 6, 1, 3), 1.0, 0.0, 3, 3),
             (256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7), 1.0, 0.0, 2, 3)]
    for L, code, p, q, n, members in cases:
        seeds = [500 + 7 * i for i in range(members)]
        sims = [binding.Sim(L, sd) for sd in seeds]
        sims[0].oct_sweep(2, p, q, code)                               # member 0 starts two sweeps ahead
        binding.oct_sweep_batch(sims, n, p, q, code)
        for i in sorted(set([0, 1, members // 2, members - 1])):
            orc = Oracle(L, seeds[i])
            orc.sweep(n + (2 if i == 0 else 0), p, q, code)
            compare_state(sims[i], orc, check_heights=False)
            orc.close()
        for s_ in sims:
            s_.close()


@pytest.mark.parametrize("L", [16, 64, 1024, 4096])
def test_one_pass_observables_equal_the_three_separate_calls_and_the_oracle(L):
    """oct_observe: any combination of the W^2, C_h and C_s sums in ONE pass over lattice + snapshot."""
    h, h2 = sf.separable_surface(L, 5, 40), sf.separable_surface(L, 105, -3)
    lat = torch.from_numpy(sf.pack_heights(h).view(np.int32).reshape(-1)).cuda()
    sim = binding.Sim(L, 0, lattice=lat)
    sim.oct_set_state(11, 40, 9)
    snap = torch.from_numpy(sf.pack_heights(h2).view(np.int32).reshape(-1)).cuda()
    anchor = torch.tensor([-3, 4], dtype=torch.int64, device="cuda")
    orc = Oracle(L, 0); orc.set_lattice(sf.pack_heights(h), h00=40, net=9)
    osn = Oracle(L, 0); osn.set_lattice(sf.pack_heights(h2), h00=-3, net=4)
    want = {1: orc.sums(), 2: orc.autocorr_sums(osn), 4: orc.slope_autocorr_sums(osn)}
    sl = {1: slice(0, 4), 2: slice(4, 9), 4: slice(9, 15)}
    for what in range(1, 8):
        out = [int(v) for v in sim.oct_observe(what, snap, anchor).cpu().numpy()]
        for bit in (1, 2, 4):
            got = tuple(out[sl[bit]])
            assert got == (want[bit] if what & bit else (0,) * len(want[bit])), (L, what, bit)
        assert out[15] == 0
    assert tuple(int(v) for v in sim.oct_width2().cpu().numpy()) == want[1]
    assert tuple(int(v) for v in sim.oct_autocorr(snap, anchor).cpu().numpy()) == want[2]
    assert tuple(int(v) for v in sim.oct_slope_autocorr(snap).cpu().numpy()) == want[4]
    with pytest.raises(binding.OctError):
        sim.oct_observe(2, None, None)
    with pytest.raises(binding.OctError):
        sim.oct_observe(8, snap, anchor)
    host = np.zeros(16, dtype=np.int64)
    sim.oct_fetch(sim.oct_observe(7, snap, anchor), host.ctypes.data, 128)
    assert tuple(host[:4]) == want[1] and tuple(host[9:15]) == want[4]
    sim.close(); orc.close(); osn.close()


def test_batch_observables_equal_the_single_calls_and_the_oracle():
    """oct_observe_batch (one launch set for an ensemble, PAPER.md:200 / :232 sample sizes) gives every member exactly the sums
    its own oct_observe gives, which are the oracle's; more members than one launch holds, and every `what`."""
    L, n = 256, 67
    code = wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)
    sims = [binding.Sim(L, 100 + i) for i in range(n)]
    binding.oct_sweep_batch(sims, 3, 1.0, 0.0, code)
    snaps = [s.oct_snapshot() for s in sims]
    binding.oct_sweep_batch(sims, 2, 1.0, 0.0, code)
    for what in (1, 2, 4, 7):
        need = what & 6
        got = binding.oct_observe_batch(sims, what, [sn[0] for sn in snaps] if need else None,
                                        [sn[1] for sn in snaps] if what & 2 else None).cpu().numpy()
        for i in (0, 1, 63, 64, n - 1):
            one = sims[i].oct_observe(what, snaps[i][0] if need else None, snaps[i][1] if what & 2 else None).cpu().numpy()
            assert (got[i] == one).all(), (what, i)
    for i in (0, 65):
        o = Oracle(L, 100 + i)
        o.sweep(3, 1.0, 0.0, code)
        osnap = o.clone()
        o.sweep(2, 1.0, 0.0, code)
        assert tuple(int(v) for v in got[i][:4]) == o.sums()
        assert tuple(int(v) for v in got[i][4:9]) == o.autocorr_sums(osnap)
        assert tuple(int(v) for v in got[i][9:15]) == o.slope_autocorr_sums(osnap)
        o.close(); osnap.close()
    with pytest.raises(binding.OctError):
        binding.oct_observe_batch(sims, 2, None, None)
    for s in sims:
        s.close()
