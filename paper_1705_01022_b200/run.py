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
import time

from . import binding, workloads as wl


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
    ap.add_argument("--seeds", type=int, default=1, help="ensemble: run seeds seed .. seed+seeds-1 concurrently (one stream each) and average")
    ap.add_argument("--log2D", type=int, default=6)
    ap.add_argument("--tcx", type=int, default=1)
    ap.add_argument("--tcy", type=int, default=1)
    ap.add_argument("--dev", type=int, default=wl.DEV_DTR)
    ap.add_argument("--blk", type=int, default=wl.BLK_DB)
    ap.add_argument("--per-decade", type=int, default=8)
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)

    import torch
    L, N = args.L, args.L * args.L
    code = wl.scheme_code(args.dev, args.blk, args.log2D, args.tcx, args.tcy)
    grid = log_grid(args.mcs, args.per_decade)
    if args.snap:
        grid = sorted(set(grid) | {args.snap} | {args.snap + t for t in log_grid(args.mcs - args.snap, args.per_decade) if args.snap + t <= args.mcs})

    # one simulation per seed, each on its own stream: small lattices do not fill the GPU alone, so the
    # members of an ensemble run concurrently (they share nothing; every call only enqueues work)
    seeds = list(range(args.seed, args.seed + args.seeds))
    runs = []
    for sd in seeds:
        stream = torch.cuda.Stream() if len(seeds) > 1 else torch.cuda.current_stream()
        with torch.cuda.stream(stream):
            sim = binding.Sim(L, sd)
        runs.append({"seed": sd, "sim": sim, "stream": stream, "snap": None, "anchor": None, "rows": [],
                     "w2": torch.empty(4, dtype=torch.int64, device=sim.device),
                     "ch": torch.empty(5, dtype=torch.int64, device=sim.device),
                     "cs": torch.empty(6, dtype=torch.int64, device=sim.device)})
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    t_now = 0
    for t in grid:
        for r in runs:                                           # enqueue on every member's stream ...
            sim, st = r["sim"], r["stream"]
            sim.oct_sweep(t - t_now, args.p, args.q, code, stream=st)
            sim.oct_width2(r["w2"], stream=st)
            if args.snap and t == args.snap:
                with torch.cuda.stream(st):
                    r["snap"], r["anchor"] = sim.oct_snapshot(stream=st)
            if r["snap"] is not None:
                sim.oct_autocorr(r["snap"], r["anchor"], r["ch"], stream=st)
                sim.oct_slope_autocorr(r["snap"], r["cs"], stream=st)
        t_now = t
        torch.cuda.synchronize()                                 # ... then read the integer sums back
        for r in runs:
            S1, S2, c, net = (int(v) for v in r["w2"].cpu())
            row = {"t": t, "w2": binding.oct_w2_from_sums(L, S1, S2), "mean_h": c + S1 / N, "net": net}
            if r["snap"] is not None:
                St, Ss, Sts, _, _ = (int(v) for v in r["ch"].cpu())
                xx, yy, xt, yt, xs, ys = (int(v) for v in r["cs"].cpu())
                row["c_h"] = binding.oct_c_from_sums(L, St, Ss, Sts)
                row["c_s"] = binding.oct_cs_from_sums(2 * N, xx + yy, xt + yt, xs + ys)
            r["rows"].append(row)
    wall = time.perf_counter() - wall0

    for r in runs:
        prev = None
        for row in r["rows"]:                                    # Eq. (8): effective exponents between grid points
            if prev is not None:
                row["beta_eff"] = (eff_exponent(row["w2"], row["t"], prev["w2"], prev["t"]) or 0.0) / 2 if row["t"] > 1 else None
                if "c_h" in row and "c_h" in prev and args.snap and prev["t"] > args.snap:
                    row["lambda_h_over_z_eff"] = -(eff_exponent(row["c_h"], row["t"] / args.snap, prev["c_h"], prev["t"] / args.snap) or float("nan"))
            prev = row
        r["sim"].close()

    fmt = lambda d: " ".join(f"{k}={v:.6g}" if isinstance(v, float) else f"{k}={v}" for k, v in d.items())
    total = len(seeds) * args.mcs * N
    result = {"L": L, "p": args.p, "q": args.q, "seeds": seeds, "scheme": wl.scheme_name(code), "mcs": args.mcs, "snap": args.snap,
              "wall_s": wall, "attempts_per_s_incl_observables": total / wall}
    if len(seeds) == 1:
        result["seed"] = seeds[0]
        result["rows"] = runs[0]["rows"]
        for row in result["rows"]:
            print(fmt(row))
    else:
        result["runs"] = [{"seed": r["seed"], "rows": r["rows"]} for r in runs]
        result["ensemble"] = ensemble_mean([r["rows"] for r in runs])
        for row in result["ensemble"]:
            print("ensemble " + fmt(row))
    print(f"# {wl.scheme_name(code)} L={L}: {len(seeds)} x {args.mcs} MCS in {wall:.1f} s = {total / wall:.4g} attempts/s including the observables")
    if args.out:
        with open(args.out, "w") as f:
            json.dump(result, f, indent=1)
    return result


if __name__ == "__main__":
    main()
