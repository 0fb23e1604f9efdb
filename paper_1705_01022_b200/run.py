"""Run one simulation of the paper's kind on the GPU and print its observables on a log-spaced time grid.

    python -m paper_1705_01022_b200.run --L 65536 --mcs 10000 --snap 1000 --log2D 6 --out run.json

This is the driver a user of the library needs for the workloads of BASELINE.json configs 4 and 5: a
growth run from the flat state (p = 1, q = 0) that records the roughness W^2(t) (Eq. (3) :61),
the mean height, and -- after a waiting-time snapshot at t = s (:80) -- the aging autocorrelations
C_h(t,s) (Eq. (6) :92-98) and C_s(t,s) (:85-88).  Effective exponents follow Eq. (8) :108-112:
e_eff = ln(E(t)/E(t')) / ln(t/t') between consecutive grid points (2 beta_eff from W^2, -lambda/z from C).
Everything numerical happens in the CUDA kernels behind the C ABI; this file only schedules calls and
divides integer sums.
"""
from __future__ import annotations

import argparse
import json
import math
import sys
import time

from . import binding, workloads as wl


def _strip(argv, flags):
    """argv without the given `--flag value` pairs"""
    out, skip = [], False
    for a in argv:
        if skip:
            skip = False
        elif a in flags:
            skip = True
        elif any(a.startswith(f + "=") for f in flags):
            pass
        else:
            out.append(a)
    return out


def log_grid(t_max: int, per_decade: int, t_min: int = 1):
    pts, k = set(), 0
    while True:
        t = int(round(t_min * 10 ** (k / per_decade)))
        if t > t_max:
            break
        pts.add(max(t, t_min))
        k += 1
    pts.add(t_max)
    return sorted(pts)


def eff_exponent(e1, t1, e0, t0):
    if e0 is None or e1 is None or e0 <= 0 or e1 <= 0 or t0 <= 0 or t1 <= t0:
        return None
    return math.log(e1 / e0) / math.log(t1 / t0)


def ensemble_mean(runs, keys=("w2", "mean_h", "c_h", "c_s")):
    """Mean and standard error over independent runs (seeds) of the per-run observables, grid point by grid
    point -- the paper's ensemble average (R8: <.> inside a run is spatial, the sample mean
    over runs is formed afterwards).  `runs` = list of row lists sharing one time grid."""
    out = []
    for rows in zip(*runs):
        t = rows[0]["t"]
        assert all(r["t"] == t for r in rows)
        rec = {"t": t, "n": len(rows)}
        for k in keys:
            vals = [r[k] for r in rows if k in r]
            if len(vals) != len(rows):
                continue
            m = sum(vals) / len(vals)
            rec[k] = m
            rec[k + "_sem"] = math.sqrt(sum((v - m) ** 2 for v in vals) / (len(vals) * (len(vals) - 1))) if len(vals) > 1 else None
        out.append(rec)
    prev = None
    for r in out:                                                # Eq. (8) on the ensemble means
        if prev is not None and r["t"] > 1:
            e = eff_exponent(r["w2"], r["t"], prev["w2"], prev["t"])
            r["beta_eff"] = None if e is None else e / 2
        prev = r
    return out


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--L", type=int, default=1 << 16)
    ap.add_argument("--mcs", type=int, default=10_000)
    ap.add_argument("--snap", type=int, default=0, help="waiting time s of the aging snapshot (0: none)")
    ap.add_argument("--p", type=float, default=1.0)
    ap.add_argument("--q", type=float, default=0.0)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--seeds", type=int, default=1, help="ensemble: run seeds seed .. seed+seeds-1 one after the other and average")
    ap.add_argument("--log2D", type=int, default=6)
    ap.add_argument("--tcx", type=int, default=1)
    ap.add_argument("--tcy", type=int, default=1)
    ap.add_argument("--dev", type=int, default=wl.DEV_DTR)
    ap.add_argument("--blk", type=int, default=wl.BLK_DB)
    ap.add_argument("--per-decade", type=int, default=8)
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)
    if args.seeds > 1:
        runs = []
        for sd in range(args.seed, args.seed + args.seeds):
            sub = list(argv if argv is not None else sys.argv[1:])
            one = main(_strip(sub, ("--seeds", "--seed", "--out")) + ["--seed", str(sd)])
            runs.append(one["rows"])
        ens = ensemble_mean(runs)
        for r in ens:
            print("ensemble " + " ".join(f"{k}={v:.6g}" if isinstance(v, float) else f"{k}={v}" for k, v in r.items()))
        if args.out:
            with open(args.out, "w") as f:
                json.dump({"seeds": list(range(args.seed, args.seed + args.seeds)), "ensemble": ens}, f, indent=1)
        return {"ensemble": ens}

    import torch
    L, N = args.L, args.L * args.L
    code = wl.scheme_code(args.dev, args.blk, args.log2D, args.tcx, args.tcy)
    sim = binding.Sim(L, args.seed)
    grid = log_grid(args.mcs, args.per_decade)
    if args.snap:
        grid = sorted(set(grid) | {args.snap} | {args.snap + t for t in log_grid(args.mcs - args.snap, args.per_decade) if args.snap + t <= args.mcs})
    w2_dev = torch.empty(4, dtype=torch.int64, device=sim.device)
    ch_dev = torch.empty(5, dtype=torch.int64, device=sim.device)
    cs_dev = torch.empty(6, dtype=torch.int64, device=sim.device)
    snap = anchor = None
    rows, t_now = [], 0
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    for t in grid:
        sim.oct_sweep(t - t_now, args.p, args.q, code)
        t_now = t
        sim.oct_width2(w2_dev)
        if args.snap and t == args.snap:
            snap, anchor = sim.oct_snapshot()
        S1, S2, c, net = (int(v) for v in w2_dev.cpu())
        row = {"t": t, "w2": binding.oct_w2_from_sums(L, S1, S2), "mean_h": c + S1 / N, "net": net}
        if snap is not None:
            sim.oct_autocorr(snap, anchor, ch_dev)
            sim.oct_slope_autocorr(snap, cs_dev)
            St, Ss, Sts, _, _ = (int(v) for v in ch_dev.cpu())
            xx, yy, xt, yt, xs, ys = (int(v) for v in cs_dev.cpu())
            row["c_h"] = binding.oct_c_from_sums(L, St, Ss, Sts)
            row["c_s"] = binding.oct_cs_from_sums(2 * N, xx + yy, xt + yt, xs + ys)
        rows.append(row)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0

    prev = None
    for r in rows:                                               # Eq. (8): effective exponents between grid points
        if prev is not None:
            r["beta_eff"] = (eff_exponent(r["w2"], r["t"], prev["w2"], prev["t"]) or 0.0) / 2 if r["t"] > 1 else None
            if "c_h" in r and "c_h" in prev and args.snap and prev["t"] > args.snap:
                r["lambda_h_over_z_eff"] = -(eff_exponent(r["c_h"], r["t"] / args.snap, prev["c_h"], prev["t"] / args.snap) or float("nan"))
        prev = r
    result = {"L": L, "p": args.p, "q": args.q, "seed": args.seed, "scheme": wl.scheme_name(code), "mcs": args.mcs,
              "snap": args.snap, "wall_s": wall, "attempts_per_s_incl_observables": args.mcs * N / wall, "rows": rows}
    for r in rows:
        print(" ".join(f"{k}={v:.6g}" if isinstance(v, float) else f"{k}={v}" for k, v in r.items()))
    print(f"# {wl.scheme_name(code)} L={L}: {args.mcs} MCS in {wall:.1f} s = {args.mcs * N / wall:.4g} attempts/s including the observables")
    if args.out:
        with open(args.out, "w") as f:
            json.dump(result, f, indent=1)
    sim.close()
    return result


if __name__ == "__main__":
    main()
