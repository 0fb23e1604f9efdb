"""Run simulations of the paper's kind on the GPU and print their observables on a log-spaced time grid.

    python -m paper_1705_01022_b200.run --L 65536 --mcs 10000 --snap 1000 --log2D 6 --out run.json
    python -m paper_1705_01022_b200.run --L 1024 --mcs 2000 --snap 100 --seeds 32 --dev 3 --blk 2      # ensemble

This is the driver a user of the library needs for the workloads of BASELINE.json: a growth run from the flat state
(p = 1, q = 0) that records the roughness W^2(t) (Eq. (3) :61), the mean height, and -- after a waiting-time
snapshot at t = s (:80) -- the aging autocorrelations C_h(t,s) (Eq. (6) :92-98) and C_s(t,s) (:85-88); all sums of one
measurement point come from ONE pass over the lattice (oct_observe; oct_observe_batch for an ensemble: three launches
per 64 members).  `--seeds N` runs an ensemble of N independent
lattices in the same kernel launches (oct_sweep_batch; the paper's curves are means over n = 20 ... 4367 runs, :200,
:232, :248) and reports mean +- s.e.m.  Effective exponents follow Eq. (8) :108-112 between consecutive grid points,
e_eff = ln(E(t)/E(t')) / ln(t/t') (2 beta_eff from W^2, -lambda/z from C), with propagated 1-sigma errors (Fig. 6
caption :248).  Under the dead-border device layers one sweep lasts (1 - N_border/N) MCS (Eq. (9) :137, reading R9):
the time axis `t` is physical time, `sweeps` counts oct_sweep units.
Everything numerical happens in the CUDA kernels behind the C ABI; this file only schedules calls and divides integer sums.
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
    """Eq. (8): ln(e1/e0) / ln(t1/t0), or None where it is not defined."""
    if e0 is None or e1 is None or e0 <= 0 or e1 <= 0 or t0 <= 0 or t1 <= t0:
        return None
    return math.log(e1 / e0) / math.log(t1 / t0)


def eff_exponent_err(e1, s1, t1, e0, s0, t0):
    """1-sigma error of eff_exponent propagated from the standard errors s1, s0 of e1, e0 (taken as independent):
    sqrt((s1/e1)^2 + (s0/e0)^2) / ln(t1/t0)."""
    if None in (e0, e1, s0, s1) or e0 <= 0 or e1 <= 0 or t0 <= 0 or t1 <= t0:
        return None
    return math.sqrt((s1 / e1) ** 2 + (s0 / e0) ** 2) / math.log(t1 / t0)


def _mean_sem(vals):
    m = sum(vals) / len(vals)
    if len(vals) < 2:
        return m, None
    return m, math.sqrt(sum((v - m) ** 2 for v in vals) / (len(vals) * (len(vals) - 1)))


def ensemble_mean(runs, keys=("w2", "mean_h", "c_h", "c_s"), snap_t=None):
    """Mean and standard error over independent runs (seeds) of the per-run observables, grid point by grid point -- the
    paper's ensemble average (R8: <.> inside a run is spatial, the sample mean over runs is formed
    afterwards) -- and the effective exponents of Eq. (8) on the means, each with (a) the error propagated from the two
    standard errors (`*_err`, the paper's "propagated 1 sigma error bars", :248) and (b) the standard error of the
    per-run exponents (`*_sem`, which knows that consecutive points of one run are correlated).
    `runs` = list of row lists sharing one time grid; snap_t = physical time of the aging snapshot (for lambda/z)."""
    out = []
    for rows in zip(*runs):
        t = rows[0]["t"]
        assert all(r["t"] == t for r in rows)
        rec = {"t": t, "n": len(rows)}
        if "sweeps" in rows[0]:
            rec["sweeps"] = rows[0]["sweeps"]
        for k in keys:
            vals = [r[k] for r in rows if k in r]
            if len(vals) != len(rows):
                continue
            rec[k], rec[k + "_sem"] = _mean_sem(vals)
        out.append(rec)
    for i in range(1, len(out)):
        r, pv = out[i], out[i - 1]
        if r["t"] <= pv["t"] or pv["t"] <= 0:
            continue
        e = eff_exponent(r.get("w2"), r["t"], pv.get("w2"), pv["t"])
        if e is not None:
            r["beta_eff"] = e / 2
            err = eff_exponent_err(r["w2"], r.get("w2_sem"), r["t"], pv["w2"], pv.get("w2_sem"), pv["t"])
            r["beta_eff_err"] = None if err is None else err / 2
            per_run = [eff_exponent(a[i]["w2"], r["t"], a[i - 1]["w2"], pv["t"]) for a in runs]
            if all(v is not None for v in per_run):
                r["beta_eff_sem"] = None if len(per_run) < 2 else _mean_sem([v / 2 for v in per_run])[1]
        if snap_t and "c_h" in r and "c_h" in pv and pv["t"] > snap_t:
            e = eff_exponent(r["c_h"], r["t"] / snap_t, pv["c_h"], pv["t"] / snap_t)
            if e is not None:
                r["lambda_h_over_z_eff"] = -e
                r["lambda_h_over_z_eff_err"] = eff_exponent_err(r["c_h"], r.get("c_h_sem"), r["t"], pv["c_h"], pv.get("c_h_sem"), pv["t"])
    return out


def member_groups(n_members: int, L: int, n_groups: int = 0):
    """Split an ensemble into groups that run on their own CUDA streams (`--streams`).  0 = one group: oct_sweep_batch
    itself runs the two halves of its members side by side (a launch of a few thousand domains leaves the GPU partly idle
    while its last domains finish; the other half fills that tail), so more groups only help to overlap the per-member
    observables of measurement-heavy runs."""
    if n_groups <= 0:
        n_groups = 1
    n_groups = max(1, min(n_groups, n_members))
    size = -(-n_members // n_groups)
    return [list(range(i, min(i + size, n_members))) for i in range(0, n_members, size)]


def simulate(L, mcs, snap, p, q, code, seeds, per_decade=8, device="cuda:0", progress=None, n_groups=0):
    """Growth / aging run of one lattice per seed (the members of a group in the same launches, groups on concurrent
    streams).  Returns (runs, wall seconds): runs[i] = rows of seed i on the common grid, each
    {sweeps, t, w2, mean_h, net[, c_h, c_s]}."""
    import torch
    N = L * L
    dt = binding.oct_time_per_sweep(L, code)                     # Eq. (9): physical MCS per sweep (1 for DT / DTr)
    grid = log_grid(mcs, per_decade)
    if snap:
        grid = sorted(set(grid) | {snap} | {snap + t for t in log_grid(mcs - snap, per_decade) if snap + t <= mcs})
    sims = [binding.Sim(L, sd, device=device) for sd in seeds]
    outs = torch.empty((len(sims), 16), dtype=torch.int64, device=sims[0].device)     # member i's sums in row i
    snaps = [None] * len(sims)
    rows = [[] for _ in sims]
    groups = member_groups(len(sims), L, n_groups)
    streams = [torch.cuda.current_stream(sims[0].device)] if len(groups) == 1 else [torch.cuda.Stream(sims[0].device) for _ in groups]
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    t_now = 0
    for t in grid:
        for members, stream in zip(groups, streams):
            if len(members) == 1:
                sims[members[0]].oct_sweep(t - t_now, p, q, code, stream=stream)
            else:
                binding.oct_sweep_batch([sims[i] for i in members], t - t_now, p, q, code, stream=stream)
        for members, stream in zip(groups, streams):
            if snap and t == snap:
                for i in members:
                    snaps[i] = sims[i].oct_snapshot(stream=stream)
            aged = snaps[members[0]] is not None
            what = (binding.OCT_OBS_W2 | binding.OCT_OBS_CH | binding.OCT_OBS_CS) if aged else binding.OCT_OBS_W2
            binding.oct_observe_batch([sims[i] for i in members], what, [snaps[i][0] for i in members] if aged else None,
                                      [snaps[i][1] for i in members] if aged else None, outs[members[0]:members[-1] + 1], stream=stream)
        t_now = t
        torch.cuda.synchronize()                                 # every group has delivered its sums
        host = outs.cpu().numpy()                                # one read-back per grid point
        for i in range(len(sims)):
            o = [int(v) for v in host[i]]
            row = {"sweeps": t, "t": t * dt, "w2": binding.oct_w2_from_sums(L, o[0], o[1]), "mean_h": o[2] + o[0] / N, "net": o[3]}
            if snaps[i] is not None:
                row["c_h"] = binding.oct_c_from_sums(L, o[4], o[5], o[6])
                row["c_s"] = binding.oct_cs_from_sums(2 * N, o[9] + o[10], o[11] + o[12], o[13] + o[14])
            rows[i].append(row)
        if progress:
            progress(t)
    wall = time.perf_counter() - wall0
    for sim in sims:
        sim.close()
    return rows, wall


def add_effective_exponents(rows, snap_t):
    prev = None
    for row in rows:                                             # Eq. (8) between consecutive grid points
        if prev is not None and row["t"] > prev["t"] > 0:
            e = eff_exponent(row["w2"], row["t"], prev["w2"], prev["t"])
            row["beta_eff"] = None if e is None else e / 2
            if snap_t and "c_h" in row and "c_h" in prev and prev["t"] > snap_t:
                e = eff_exponent(row["c_h"], row["t"] / snap_t, prev["c_h"], prev["t"] / snap_t)
                row["lambda_h_over_z_eff"] = None if e is None else -e
        prev = row


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--L", type=int, default=1 << 16)
    ap.add_argument("--mcs", type=int, default=10_000, help="number of sweeps (= MCS for DT / DTr device layers)")
    ap.add_argument("--snap", type=int, default=0, help="waiting time s of the aging snapshot, in sweeps (0: none)")
    ap.add_argument("--p", type=float, default=1.0)
    ap.add_argument("--q", type=float, default=0.0)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--seeds", type=int, default=1, help="ensemble: seeds seed .. seed+seeds-1, all members in each kernel launch")
    ap.add_argument("--log2D", type=int, default=6)
    ap.add_argument("--tcx", type=int, default=1)
    ap.add_argument("--tcy", type=int, default=1)
    ap.add_argument("--dev", type=int, default=wl.DEV_DTR)
    ap.add_argument("--blk", type=int, default=wl.BLK_DB)
    ap.add_argument("--ka", type=int, default=0, help="dead-border layers: t_async = 2^-ka MCS (PAPER.md:204-206)")
    ap.add_argument("--w", type=int, default=0, help="dead-border layers: border width in sites, 0 = the scheme's own (PAPER.md:202, :208)")
    ap.add_argument("--per-decade", type=int, default=8)
    ap.add_argument("--streams", type=int, default=0, help="ensemble: groups of members on concurrent CUDA streams (0: choose)")
    ap.add_argument("--out", default="")
    args = ap.parse_args(argv)

    L, N = args.L, args.L * args.L
    code = wl.scheme_code(args.dev, args.blk, args.log2D, args.tcx, args.tcy, args.ka, args.w)
    seeds = list(range(args.seed, args.seed + args.seeds))
    runs, wall = simulate(L, args.mcs, args.snap, args.p, args.q, code, seeds, args.per_decade, n_groups=args.streams)
    dt = binding.oct_time_per_sweep(L, code)
    snap_t = args.snap * dt
    for rows in runs:
        add_effective_exponents(rows, snap_t)

    fmt = lambda d: " ".join(f"{k}={v:.6g}" if isinstance(v, float) else f"{k}={v}" for k, v in d.items())   # noqa: E731
    total = len(seeds) * args.mcs * N
    result = {"L": L, "p": args.p, "q": args.q, "seeds": seeds, "scheme": wl.scheme_name(code), "mcs": args.mcs, "snap": args.snap,
              "mcs_per_sweep": dt, "wall_s": wall, "attempts_per_s_incl_observables": total / wall}
    if len(seeds) == 1:
        result["seed"] = seeds[0]
        result["rows"] = runs[0]
        for row in result["rows"]:
            print(fmt(row))
    else:
        result["runs"] = [{"seed": sd, "rows": rows} for sd, rows in zip(seeds, runs)]
        result["ensemble"] = ensemble_mean(runs, snap_t=snap_t)
        for row in result["ensemble"]:
            print("ensemble " + fmt(row))
    print(f"# {wl.scheme_name(code)} L={L}: {len(seeds)} x {args.mcs} sweeps in {wall:.1f} s = {total / wall:.4g} attempts/s including the observables")
    if args.out:
        with open(args.out, "w") as f:
            json.dump(result, f, indent=1)
    return result


if __name__ == "__main__":
    main()
