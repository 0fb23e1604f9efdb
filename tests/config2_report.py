"""BASELINE config 2 as the paper poses it (Sec. 4.1.1, Fig. 3): every DD scheme the paper defines
against the oracle's TRUE random-sequential dynamics, L = 1024, p = 1, q = 0, flat start, 2000 MCS, seeds 1..8:
W^2(t) on a log grid and the autocorrelations C_h(t,s), C_s(t,s) at s = 100 and 200 (the stored ensemble is 32 seeds).

The RS reference is tests/golden/rs_L1024.txt (exact integer sums written by tests/golden/make_rs_golden.py from
oracle/ only).  The DD schemes run on the GPU through the C ABI, all eight seeds in the same launches (oct_sweep_batch).
Dead-border schemes are compared at equal PHYSICAL time: one DB / cDB sweep lasts (1 - N_border/N) MCS (Eq. (9) :137,
reading R9), so a grid time t is reached after round(t / oct_time_per_sweep) sweeps.

    python tests/config2_report.py            # markdown table (needs a B200); tests/test_gpu_config2.py asserts on the same numbers
"""
from __future__ import annotations

import math
import os
import sys
from fractions import Fraction

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L, P, Q, WAITS, LOG2D = 1024, 1.0, 0.0, (100, 200), 7
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "rs_L1024.txt")
# seeds of the stored RS runs: BASELINE config 2 asks for 1..8; the file holds 1..32 so that the C_s plateaus the paper
# describes (a few 1e-4 at this size) stand several standard errors above the noise
SEEDS = tuple(sorted({int(l.split()[1]) for l in open(GOLDEN) if l.startswith("w2 ")}))


def mean_sem(vals):
    m = sum(vals) / len(vals)
    return m, math.sqrt(sum((v - m) ** 2 for v in vals) / (len(vals) * (len(vals) - 1)))


def _w2(S1, S2):
    N = L * L
    return float(Fraction(N * S2 - S1 * S1, N * N))


def _ch(St, Ss, Sts):
    N = L * L
    return float(Fraction(N * Sts - St * Ss, N * N))


def _cs(xx, yy, xt, yt, xs, ys):
    M = 2 * L * L
    return float(Fraction(M * (xx + yy) - (xt + yt) * (xs + ys), M * M))


def rs_reference():
    """{'w2': {t: [per seed]}, 'ch': {(s,t): [...]}, 'cs': {(s,t): [...]}} from the stored oracle RS runs."""
    out = {"w2": {}, "ch": {}, "cs": {}}
    for line in open(GOLDEN):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        v = [int(x) for x in f[1:]]
        if f[0] == "w2":
            out["w2"].setdefault(v[1], []).append(_w2(v[2], v[3]))
        elif f[0] == "ch":
            out["ch"].setdefault((v[1], v[2]), []).append(_ch(v[3], v[4], v[5]))
        elif f[0] == "cs":
            out["cs"].setdefault((v[1], v[2]), []).append(_cs(*v[3:9]))
    return out


def gpu_scheme(code, grid_w2, grid_ac):
    """The same observables for DD scheme `code` on the GPU, seeds 1..8, at equal physical times."""
    import torch
    from paper_1705_01022_b200 import binding
    dt = binding.oct_time_per_sweep(L, code)
    sweeps_of = lambda t: int(round(t / dt))                                    # noqa: E731
    times = sorted(set(grid_w2) | {t for (_, t) in grid_ac})
    sims = [binding.Sim(L, sd) for sd in SEEDS]
    outs = [torch.empty(16, dtype=torch.int64, device=sims[0].device) for _ in sims]
    snaps = {s: [None] * len(sims) for s in WAITS}
    res = {"w2": {}, "ch": {}, "cs": {}}
    done = 0
    for t in times:
        n = sweeps_of(t)
        binding.oct_sweep_batch(sims, n - done, P, Q, code)
        done = n
        for s in WAITS:
            if t == s:
                snaps[s] = [sim.oct_snapshot() for sim in sims]
        for i, sim in enumerate(sims):
            sim.oct_observe(binding.OCT_OBS_W2, None, None, outs[i])
        host = torch.stack(outs).cpu().numpy()
        if t in grid_w2:
            res["w2"][t] = [_w2(int(h[0]), int(h[1])) for h in host]
        for s in WAITS:
            if (s, t) in grid_ac:
                for i, sim in enumerate(sims):
                    sim.oct_observe(binding.OCT_OBS_CH | binding.OCT_OBS_CS, snaps[s][i][0], snaps[s][i][1], outs[i])
                host = torch.stack(outs).cpu().numpy()
                res["ch"][(s, t)] = [_ch(int(h[4]), int(h[5]), int(h[6])) for h in host]
                res["cs"][(s, t)] = [_cs(*[int(v) for v in h[9:15]]) for h in host]
    for sim in sims:
        sim.close()
    return res


def schemes():
    from paper_1705_01022_b200 import workloads as wl
    sc = wl.scheme_code
    return [("DTrDB", sc(wl.DEV_DTR, wl.BLK_DB, LOG2D)), ("DTrDT", sc(wl.DEV_DTR, wl.BLK_DT, LOG2D)),
            ("DTrDB TC=2,2", sc(wl.DEV_DTR, wl.BLK_DB, LOG2D, 2, 2)),
            ("DT.DT", sc(wl.DEV_DT, wl.BLK_DT, LOG2D)), ("cDB.DT", sc(wl.DEV_CDB, wl.BLK_DT, LOG2D)),
            ("DB.DT", sc(wl.DEV_DB, wl.BLK_DT, LOG2D)), ("DBh.DT", sc(wl.DEV_DBH, wl.BLK_DT, LOG2D)),
            ("DB.DT tasync=1/4", sc(wl.DEV_DB, wl.BLK_DT, LOG2D, 1, 1, 2, 0)), ("DB.DT w=1", sc(wl.DEV_DB, wl.BLK_DT, LOG2D, 1, 1, 0, 1)),
            ("DB.DT w=1 tasync=1/4", sc(wl.DEV_DB, wl.BLK_DT, LOG2D, 1, 1, 2, 1))]


def late_mean(cs, s, ratio_min=6):
    """ensemble mean and standard error of C_s(t,s) averaged over the late grid points t >= ratio_min * s, per seed first"""
    keys = sorted(k for k in cs if k[0] == s and k[1] >= ratio_min * s)
    per_seed = [sum(cs[k][i] for k in keys) / len(keys) for i in range(len(cs[keys[0]]))]
    return mean_sem(per_seed)


def compare(rs, dd):
    """Deviations of a DD scheme from RS: W^2 at t = 100 and 2000 (relative, and in combined standard errors), C_h(t,s)
    at t/s = 2 and 10 (s = 100) and t/s = 2 (s = 200), late-time C_s plateau for both waiting times."""
    rec = {}
    for t in (100, 1024, 2000):
        (a, sa), (b, sb) = mean_sem(dd["w2"][t]), mean_sem(rs["w2"][t])
        rec[f"w2_{t}"] = {"dd": a, "rs": b, "rel": a / b - 1, "sigmas": (a - b) / math.hypot(sa, sb)}
    for (s, t) in ((100, 200), (100, 1200), (200, 400), (200, 2000)):
        (a, sa), (b, sb) = mean_sem(dd["ch"][(s, t)]), mean_sem(rs["ch"][(s, t)])
        rec[f"ch_{s}_{t}"] = {"dd": a, "rs": b, "rel": a / b - 1, "sigmas": (a - b) / math.hypot(sa, sb)}
    for s in WAITS:
        (a, sa), (b, sb) = late_mean(dd["cs"], s), late_mean(rs["cs"], s)
        rec[f"cs_late_{s}"] = {"dd": a, "dd_sem": sa, "rs": b, "rs_sem": sb, "sigmas": (a - b) / math.hypot(sa, sb)}
    return rec


def main():
    rs = rs_reference()
    grid_w2 = sorted(rs["w2"])
    grid_ac = sorted(rs["ch"])
    print(f"RS (oracle, tests/golden/rs_L1024.txt), L={L}, seeds {SEEDS[0]}..{SEEDS[-1]}; DD schemes on the GPU, D={1 << LOG2D}, same seeds\n")
    print("| scheme | W2(100) rel / sigma | W2(2000) rel / sigma | C_h(200,100) rel / sigma | C_h(1200,100) rel / sigma | C_h(2000,200) rel / sigma | late C_s, s=100 (mean +- sem; sigma vs RS) | late C_s, s=200 |")
    print("|---|---|---|---|---|---|---|---|")
    a, sa = late_mean(rs["cs"], 100)
    b, sb = late_mean(rs["cs"], 200)
    print(f"| RS | {mean_sem(rs['w2'][100])[0]:.4f} | {mean_sem(rs['w2'][2000])[0]:.4f} | {mean_sem(rs['ch'][(100, 200)])[0]:.4f} | {mean_sem(rs['ch'][(100, 1200)])[0]:.4f} | "
          f"{mean_sem(rs['ch'][(200, 2000)])[0]:.4f} | {a:+.2e} +- {sa:.1e} | {b:+.2e} +- {sb:.1e} |")
    for name, code in schemes():
        c = compare(rs, gpu_scheme(code, grid_w2, grid_ac))
        f = lambda k: f"{c[k]['rel']:+.2%} / {c[k]['sigmas']:+.1f}"                # noqa: E731
        g = lambda k: f"{c[k]['dd']:+.2e} +- {c[k]['dd_sem']:.1e}; {c[k]['sigmas']:+.1f}"   # noqa: E731
        print(f"| {name} | {f('w2_100')} | {f('w2_2000')} | {f('ch_100_200')} | {f('ch_100_1200')} | {f('ch_200_2000')} | {g('cs_late_100')} | {g('cs_late_200')} |")


if __name__ == "__main__":
    main()
