"""GPU parity at BASELINE.json's full sizes (configs 4 and 5: L = 2^16 and 2^17), in the launch
configuration bench.py times.

The oracle cannot sweep 2^32 sites in seconds, but it does not have to: a domain sweep depends only on
its own window, so running only the domains that meet a box reproduces the full run inside the box
shrunk by 4(D+2) sites per MCS (tests/test_oracle_dd.py::test_filtered_run_reproduces_the_interior pins
that tool against complete runs).  Here the GPU's lattice before and after one MCS is exported, the oracle
replays that MCS on sampled boxes (one of them across the periodic seam, one around the tracked origin
site), and the packed words inside the boxes must be identical.  Properties that hold at any size cover
the rest: slope conservation per row / column, the height-sum identity, C_h(s,s) sums == W^2 sums.
"""
import hashlib
import os

import numpy as np
import pytest

from oracle import Oracle
from paper_1705_01022_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def interior_words(x0, y0, w, h, margin, L):
    """index arrays (wy, wx) of the packed words lying entirely inside the box shrunk by `margin`"""
    xa, xb = x0 + margin, x0 + w - margin          # site range [xa, xb)
    ya, yb = y0 + margin, y0 + h - margin
    wxs = (np.arange((xa + 3) // 4, xb // 4)) % (L // 4)
    wys = (np.arange((ya + 3) // 4, yb // 4)) % (L // 4)
    assert len(wxs) > 8 and len(wys) > 8
    return np.ix_(wys, wxs)


_ORACLES = {}


def oracle_for(L, seed):
    """One oracle state per lattice size for the whole module (creating a 2^32-site state takes ~10 s)."""
    if L not in _ORACLES:
        _ORACLES[L] = Oracle(L, seed)
    return _ORACLES[L]


def replay_boxes(L, seed, code, log2D, p, q, pre, t, h00, net, post, boxes, h00_after=None):
    D = 1 << log2D
    margin = 4 * (D + 2)
    orc = oracle_for(L, seed)
    for (x0, y0) in boxes:
        w = h = 2 * margin + 4 * D
        orc.set_lattice(pre, h00=h00, net=net, t=t)
        orc.set_filter(True, x0 % L, y0 % L, w, h)
        orc.sweep(1, p, q, code)
        ix = interior_words(x0, y0, w, h, margin, L)
        got, want = post[ix], orc.lattice[ix]
        assert (got == want).all(), f"box ({x0},{y0}): {(got != want).sum()} of {got.size} words differ"
        assert (want != pre[ix]).any(), "the replayed MCS changed nothing inside the box"
        if h00_after is not None and x0 < 0 and y0 < 0:        # the box around the origin site: its tracked height too
            assert orc.h00 == h00_after
    orc.set_filter(False)


def popcount_rows(words, mask):
    """number of set bits under `mask` per word-row and per word-column (uint64 sums)"""
    v = words & np.uint32(mask)
    v = v - ((v >> 1) & np.uint32(0x55555555))
    v = (v & np.uint32(0x33333333)) + ((v >> 2) & np.uint32(0x33333333))
    v = (v + (v >> 4)) & np.uint32(0x0F0F0F0F)
    v = (v * np.uint32(0x01010101)) >> 24
    return v.sum(axis=1, dtype=np.uint64), v.sum(axis=0, dtype=np.uint64)


def check_invariants(sim, words):
    L = sim.L
    # each site row holds L/2 up-slopes in x, each site column L/2 up-slopes in y (periodic closure);
    # checked on 1024 sampled word-rows and word-columns
    pick = np.sort(np.random.default_rng(5).choice(L // 4, size=min(1024, L // 4), replace=False))
    some_rows, some_cols = words[pick, :], np.ascontiguousarray(words[:, pick])
    for j in range(4):
        rows, _ = popcount_rows(some_rows, 0x55 << (8 * j))
        assert (rows == L // 2).all()
    for i in range(4):
        _, cols = popcount_rows(some_cols, 0x02020202 << (2 * i))
        assert (cols == L // 2).all()
    S1, S2, c, net = (int(v) for v in sim.oct_width2().cpu().numpy())
    h00, net2 = sim.oct_counters()
    assert (c, net) == (h00, net2)
    assert S1 + L * L * c == L * L // 2 + 2 * net            # sum of heights: flat start + 2 per deposit
    snap, anchor = sim.oct_snapshot()
    A = [int(v) for v in sim.oct_autocorr(snap, anchor).cpu().numpy()]
    assert A[0] == A[1] == S1 and A[2] == S2 and A[3] == A[4] == c      # C_h(s,s) = W^2(s)
    del snap
    return S1, S2, c, net


@pytest.mark.parametrize("log2D,tc,p,q", [(6, 1, 1.0, 0.0), (7, 1, 1.0, 0.0), (8, 1, 1.0, 0.0),
                                          (6, 1, 0.9, 0.1),      # mixed rates at D = 64: the one-pass / three-phase decision per step
                                          (6, 2, 1.0, 0.0),      # TC=2,2: two-byte entries, two domains per warp
                                          (6, 2, 0.9, 0.1)],
                         ids=["D64", "D128", "D256", "D64-mixed", "D64-TC22", "D64-TC22-mixed"])
def test_config3_L65536_sampled_boxes(log2D, tc, p, q):
    """BASELINE config 4: L = 2^16, flat start, seed 1, DTrDB -- TC=1,1 with p = 1, q = 0 as the config states it, and the
    other shapes bench.py times at this size (`shapes`: mixed rates, TC=2,2), at the MCS it times them (24 -> 25)."""
    L, seed, kernel = 1 << 16, 1, binding.OCT_KERNEL_AUTO
    code = wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, log2D, tc, tc)
    sim = binding.Sim(L, seed)
    sim.oct_set_option(binding.OCT_OPT_KERNEL, kernel)
    # the very first MCS, from the flat state (acceptance 1/2)
    pre = sim.oct_export()
    assert (pre == 0x33CC33CC).all()
    sim.oct_sweep(1, p, q, code)
    post = sim.oct_export()
    replay_boxes(L, seed, code, log2D, p, q, pre, 0, 0, 0, post, [(1000, 2000), (L - 700, L - 900)])
    # an evolved state (what bench.py times): MCS 24 -> 25
    sim.oct_sweep(23, p, q, code)
    sim.oct_export(pre)
    h00, net = sim.oct_counters()
    sim.oct_sweep(1, p, q, code)
    sim.oct_export(post)
    D = 1 << log2D
    margin = 4 * (D + 2)
    replay_boxes(L, seed, code, log2D, p, q, pre, 24, h00, net, post,
                 [(31337, 4242), (L - 5 * D, 17 * D + 3), (-margin - 2 * D, -margin - 2 * D)], h00_after=sim.oct_counters()[0])
    S1, S2, c, net = check_invariants(sim, post)
    assert net > 0 and S2 > 0
    sim.close()
    del pre, post


def test_config4_L131072_sampled_boxes():
    """BASELINE config 5: L = 2^17 (4 GiB packed), same scheme: evolved-state MCS replayed on boxes."""
    L, seed, p, q, log2D = 1 << 17, 1, 1.0, 0.0, 6
    code = wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, log2D)
    sim = binding.Sim(L, seed)
    sim.oct_sweep(6, p, q, code)
    pre = sim.oct_export()
    h00, net = sim.oct_counters()
    sim.oct_sweep(1, p, q, code)
    post = sim.oct_export()
    replay_boxes(L, seed, code, log2D, p, q, pre, 6, h00, net, post, [(99991, 70001), (L - 300, L - 400)])
    check_invariants(sim, post)
    sim.close()


def test_config2_L4096_mixed_rates_late_time_boxes():
    """BASELINE config 3 (L = 4096, p = 0.9, q = 0.1, seed 7, DTrDB with delayed borders, D = 128) deep into the
    run: MCS 1000 -> 1001 and 4999 -> 5000 replayed by the oracle on boxes (the first 2 MCS are compared in full
    in test_gpu_parity.py); mean height and W^2 sums stay consistent with the counters all the way."""
    cfg = wl.CONFIGS[2]
    L, seed, code = cfg.L, cfg.seeds[0], cfg.scheme
    log2D = (code >> 16) & 31
    sim = binding.Sim(L, seed)
    t_now = 0
    for t in (1000, cfg.n_mcs - 1):
        sim.oct_sweep(t - t_now, cfg.p, cfg.q, code)
        pre = sim.oct_export()
        h00, net = sim.oct_counters()
        sim.oct_sweep(1, cfg.p, cfg.q, code)
        t_now = t + 1
        post = sim.oct_export()
        replay_boxes(L, seed, code, log2D, cfg.p, cfg.q, pre, t, h00, net, post, [(777, 1234), (L - 900, L - 650)])
        S1, S2, c, net2 = check_invariants(sim, post)
        assert net2 > net                                         # p > q: the surface keeps growing
    assert sim.oct_mcs() == cfg.n_mcs
    sim.close()


def test_config1_L1024_every_scheme_at_the_end_of_the_run():
    """BASELINE config 2 (L = 1024, p = 1, q = 0, 2000 MCS, D = 128): for every device-layer x block-layer scheme
    the paper defines, the last MCS of the run (1999 -> 2000) replayed by the oracle on the WHOLE lattice from the
    GPU's exported pre-state (the first MCS are compared in test_gpu_parity.py)."""
    cfg = wl.CONFIGS[1]
    L, seed = cfg.L, 1
    schemes = list(wl.ALL_SCHEMES(7)) + [wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 7), wl.scheme_code(wl.DEV_DBH, wl.BLK_DB, 7),
                                         wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7, 2, 2), wl.scheme_code(wl.DEV_DTR, wl.BLK_DB_DELAYED, 7)]
    orc = Oracle(L, seed)
    for code in schemes:
        sim = binding.Sim(L, seed)
        sim.oct_sweep(cfg.n_mcs - 1, cfg.p, cfg.q, code)
        pre = sim.oct_export()
        h00, net = sim.oct_counters()
        sim.oct_sweep(1, cfg.p, cfg.q, code)
        orc.set_lattice(pre, h00=h00, net=net, t=cfg.n_mcs - 1)
        orc.sweep(1, cfg.p, cfg.q, code)
        assert (sim.oct_export() == orc.lattice).all(), wl.scheme_name(code)
        assert sim.oct_counters() == (orc.h00, orc.net), wl.scheme_name(code)
        assert tuple(int(v) for v in sim.oct_width2().cpu().numpy()) == orc.sums(), wl.scheme_name(code)
        sim.close()
    orc.close()


# ---- whole-lattice parity at full size against stored oracle results --------------------------------------------
# tests/golden/full_<name>.txt are written by `python tests/golden/make_oracle_golden.py --full <name>` from oracle/ only
# (SHA-256 of the oracle's packed lattice + its integer sums at each checkpoint).  The CUDA path must reproduce them:
# BASELINE config 4 "the oracle checked bit-exact on the first 2 MCS" (L = 2^16), config 5 first MCS
# (L = 2^17, :232), config 3 the whole 5000-MCS mixed-rate run (p, q > 0: delayed borders, :174).
GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_full(name):
    cps, windows = [], {}
    for line in open(os.path.join(GOLDEN_DIR, f"full_{name}.txt")):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "sums_sha":
            windows[int(f[3])] = (int(f[2]), f[4])
        else:
            assert f[0] == name
            cps.append({"L": int(f[1]), "seed": int(f[2]), "p": float(f[3]), "q": float(f[4]), "code": int(f[5]), "t": int(f[6]),
                        "sha": f[7], "sums": tuple(int(v) for v in f[8:12])})
    return cps, windows


def sha_words(words):
    return hashlib.sha256(np.ascontiguousarray(words).astype("<u4", copy=False).tobytes()).hexdigest()


@pytest.mark.parametrize("name,kernel", [("c4_D64", binding.OCT_KERNEL_AUTO), ("c4_D64", binding.OCT_KERNEL_BITPACKED),
                                         ("c4_D128", binding.OCT_KERNEL_AUTO), ("c4_D256", binding.OCT_KERNEL_AUTO),
                                         ("c4_D64_TC22", binding.OCT_KERNEL_AUTO), ("c5_D64", binding.OCT_KERNEL_AUTO)])
def test_whole_lattice_equals_the_oracle_at_full_size(name, kernel):
    cps, _ = read_full(name)
    c0 = cps[0]
    sim = binding.Sim(c0["L"], c0["seed"])
    sim.oct_set_option(binding.OCT_OPT_KERNEL, kernel)
    host = np.empty((c0["L"] // 4, c0["L"] // 4), dtype=np.uint32)
    for c in cps:
        sim.oct_sweep(c["t"] - sim.oct_mcs(), c["p"], c["q"], c["code"])
        assert tuple(int(v) for v in sim.oct_width2().cpu().numpy()) == c["sums"], (name, c["t"])
        assert sim.oct_counters() == c["sums"][2:], (name, c["t"])
        assert sha_words(sim.oct_export(host)) == c["sha"], (name, c["t"])
    sim.close()


@pytest.mark.parametrize("name", ["c3_D128", "c3_D64"])
def test_config3_whole_run_equals_the_oracle(name):
    """BASELINE config 3 in full: L = 4096, p = 0.9, q = 0.1, seed 7, DTrDB (delayed borders), 5000 MCS: the lattice hash
    every 500 MCS and (S1, S2, h00, net) after EVERY MCS (W^2(t) and the mean height per MCS).  D = 128 is the config's own
    shape (four warps per domain: three phases every step); D = 64 is the shape whose domains sit in one warp, where the
    kernel decides per collective step between one pass and three phases."""
    cps, windows = read_full(name)
    assert [c["t"] for c in cps] == list(range(500, 5001, 500)) and len(windows) == len(cps)
    c0 = cps[0]
    sim = binding.Sim(c0["L"], c0["seed"])
    out = torch.empty(4, dtype=torch.int64, device=sim.device)
    for c in cps:
        t0, want = windows[c["t"]]
        assert t0 == sim.oct_mcs()
        hs, rows = hashlib.sha256(), []
        for _ in range(c["t"] - t0):
            sim.oct_sweep(1, c["p"], c["q"], c["code"])
            sim.oct_width2(out)
            rows.append(out.clone())                      # stay asynchronous; read the window back at its end
        for r in torch.stack(rows).cpu().numpy():
            hs.update(("%d %d %d %d\n" % tuple(int(v) for v in r)).encode())
        assert hs.hexdigest() == want, ("sums of MCS", t0, c["t"])
        assert tuple(int(v) for v in rows[-1].cpu().numpy()) == c["sums"], c["t"]
        assert sha_words(sim.oct_export()) == c["sha"], c["t"]
    sim.close()
