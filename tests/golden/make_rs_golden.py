#!/usr/bin/env python
"""Writes tests/golden/rs_L1024.txt: the oracle's TRUE random-sequential (RS) dynamics on BASELINE
config 2 -- L = 1024, p = 1, q = 0, flat start, 2000 MCS, seeds 1..8 -- as exact integer sums on a fixed time grid:
the W^2 sums (Eq. (3) :61) at every grid point, and the C_h (Eq. (6) :92-98) and C_s (:85-88) sums against the
waiting-time snapshots at s = 100 and s = 200.  This is the reference every DD scheme is compared with in
Sec. 4.1 (:192-210, Fig. 3).  Calls ONLY oracle/ (never the CUDA path); GPU tests and run reports read the file.

    python tests/golden/make_rs_golden.py [--workers N] [--seeds 1 8]      (about 4 minutes of one core per seed)

Line formats (integers are exact):
    w2 seed t S1 S2 h00 net
    ch seed s t St Ss Sts ct cs
    cs seed s t xx yy xt yt xs ys
"""
import argparse
import os
import sys
from concurrent.futures import ProcessPoolExecutor

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

L, P, Q, T_MAX = 1024, 1.0, 0.0, 2000
WAITS = (100, 200)
# sqrt(2)-spaced growth grid plus t/s = 1, 1.5, 2, 3, 4, 6, 8, 12, 16, 20 for both waiting times
GROWTH = (1, 2, 3, 4, 6, 8, 11, 16, 23, 32, 45, 64, 91, 128, 181, 256, 362, 512, 724, 1024, 1448, 2000)
RATIOS = (1, 1.5, 2, 3, 4, 6, 8, 12, 16, 20)
GRID = tuple(sorted(set(GROWTH) | {int(s * r) for s in WAITS for r in RATIOS if s * r <= T_MAX}))


def one_seed(seed):
    from oracle import Oracle
    o = Oracle(L, seed)
    snaps, out = {}, []
    for t in GRID:
        o.sweep_rs(t - o.t, P, Q)
        out.append("w2 %d %d %d %d %d %d" % ((seed, t) + o.sums()))
        if t in WAITS:
            snaps[t] = o.clone()
        for s, sn in sorted(snaps.items()):
            out.append("ch %d %d %d %d %d %d %d %d" % ((seed, s, t) + o.autocorr_sums(sn)))
            out.append("cs %d %d %d %d %d %d %d %d %d" % ((seed, s, t) + o.slope_autocorr_sums(sn)))
    return out


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--workers", type=int, default=2)
    ap.add_argument("--seeds", type=int, nargs=2, default=(1, 8), help="first and last seed")
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)), "rs_L1024.txt"))
    a = ap.parse_args()
    import oracle
    oracle.build()
    seeds = list(range(a.seeds[0], a.seeds[1] + 1))
    with ProcessPoolExecutor(a.workers) as ex:
        res = list(ex.map(one_seed, seeds))
    with open(a.out, "w") as f:
        f.write(f"# oracle RS dynamics, L={L} p={P} q={Q} flat start, seeds {seeds[0]}..{seeds[-1]}; formats in make_rs_golden.py\n")
        f.write("# written by `python tests/golden/make_rs_golden.py` from oracle/oct_oracle.c only\n")
        for lines in res:
            f.write("\n".join(lines) + "\n")
    print(a.out)
