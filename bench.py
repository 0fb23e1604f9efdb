#!/usr/bin/env python
"""bench.py -- throughput of the DD random-sequential sweep of the octahedron model on B200.

    python bench.py --gpus N --steps K --warmup W            (N>1: launched by torch.distributed.run)
    python bench.py --impl reference ...                     (times the CPU oracle instead)

Metric (BASELINE.json): site-update attempts per second at L = 2^16, p = 1, q = 0, scheme DTrDB
(PAPER.md:262, :276).  One *step* is one pass of the whole hot path on the resident lattice:
`--mcs-per-step` MCS of oct_sweep (4 launches per MCS), then oct_width2 and oct_autocorr against the
waiting-time snapshot.  attempts = mcs_per_step * L^2 per step (rejected attempts count, :270).
The lattice (1 GiB) is larger than L2 (126 MB), so no explicit L2 flush is needed between steps.
N > 1 runs N independent replicas (different seeds, no data-path collective: "replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "site_update_attempts_per_s"
UNIT = "attempts/s"

# Algorithmic lane-instructions per update attempt of the DTrDB sweep in the link-entry design (DESIGN.md
# section 6): Philox4x32-10 40/4 = 10, site select 5, entry load + compare 2, five stores of an accepted
# update (issued warp-wide) 5, step loop/sync 1, staging (expand + gather + moments per site) 9.
I_ALG = 32.0
# the paper's DTrDB throughput at L = 2^16, p=1, q=0 on Kepler GPUs, per GPU
PAPER_ATTEMPTS_PER_S = 9.0e9
N_SM, SMSP, LANES = 148, 4, 32


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": d.get("hbm_gbs", 6650.0), "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                c = [t.strip() for t in line.split(",")]
                if len(c) < 7:
                    continue
                try:
                    sm.append(float(c[0])); mx.append(float(c[1]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}
        return out


def time_oracle(L: int, log2D: int, n_mcs: int, seed: int):
    """The CPU oracle as it stands, single thread, on a bounded sample of the workload."""
    import oracle
    code = oracle.scheme(oracle.DEV_DTR, oracle.BLK_DB, log2D)
    o = oracle.Oracle(L, seed)
    o.sweep(1, 1.0, 0.0, code)               # leave the exactly-flat state (acceptance 0.5 -> ~0.2)
    t0 = time.perf_counter()
    o.sweep(n_mcs, 1.0, 0.0, code)
    S = o.sums()
    dt = time.perf_counter() - t0
    o.close()
    return n_mcs * L * L / dt, dt, S


def run_reference(args, rank: int, world: int):
    if rank != 0:
        return
    Ls, n_mcs = args.ref_L, args.ref_mcs
    vals, times = [], []
    for i in range(args.warmup + args.steps):
        v, dt, _ = time_oracle(Ls, min(args.log2D, 8), n_mcs, args.seed + i)
        if i >= args.warmup:
            vals.append(v); times.append(dt)
    value = sum(vals) / len(vals)
    sample = (f"per step: {n_mcs} MCS of DTrDB(D={1 << args.log2D}) incl. the W2 sums on an L={Ls} flat-start lattice "
              f"(same scheme, p, q and domain size as the L={args.L} workload; oracle/oct_oracle.c, gcc -O2, 1 thread)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": workload_config(args),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(args):
    name = "DTrDT" if getattr(args, "blk", 0) == 2 else "DTrDB"
    return {"workload": f"c3_L{args.L}: octahedron model, L={args.L} periodic, flat start, p=1 q=0, {name} TC=1,1 D={1 << args.log2D}",
            "L": args.L, "p": 1.0, "q": 0.0, "scheme": f"{name},TC=1,1,D={1 << args.log2D}", "mcs_per_step": args.mcs_per_step,
            "burn_in_mcs": args.burn_in, "l2": "inputs larger than L2 (lattice %d MiB)" % (args.L * args.L // 4 >> 20),
            "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=1 << 16)
    ap.add_argument("--log2D", type=int, default=6)
    ap.add_argument("--mcs-per-step", type=int, default=8)
    ap.add_argument("--burn-in", type=int, default=32)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--ref-L", type=int, default=4096, help="lattice edge of the oracle's timed sample")
    ap.add_argument("--ref-mcs", type=int, default=32)
    ap.add_argument("--blk", type=int, default=0, help="block layer: 0 DB (the benched DTrDB), 2 DT (DTrDT, PAPER.md:268)")
    ap.add_argument("--kernel", type=int, default=0, help="OCT_OPT_KERNEL value: 0 auto, 1 bit-packed, 2 link-entry variant B")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-heights", action="store_true", help="skip timing oct_heights (needs a 4*L*L byte buffer)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    from paper_1705_01022_b200 import binding, replicas, workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    L, M = args.L, args.mcs_per_step
    code = wl.scheme_code(wl.DEV_DTR, args.blk, args.log2D)
    seed = replicas.replica_seed(args.seed, rank)
    sim = binding.Sim(L, seed, wl.INIT_FLAT, device=f"cuda:{local_rank}")
    sim.oct_set_option(binding.OCT_OPT_KERNEL, args.kernel)
    stream = torch.cuda.current_stream()
    sim.oct_sweep(args.burn_in, 1.0, 0.0, code)            # evolved state: acceptance ~0.17 (not the flat 0.5)
    snap, anchor = sim.oct_snapshot()
    w2_out = torch.empty(4, dtype=torch.int64, device=sim.device)
    ac_out = torch.empty(5, dtype=torch.int64, device=sim.device)
    cs_out = torch.empty(6, dtype=torch.int64, device=sim.device)

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        sim.oct_sweep(M, 1.0, 0.0, code)
        if ev:
            ev[1].record(stream)
        sim.oct_width2(w2_out)
        sim.oct_autocorr(snap, anchor, ac_out)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    n0 = sim.oct_launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        step(evs[i])
    e1.record(stream)
    barrier()
    launches = sim.oct_launch_count() - n0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = e0.elapsed_time(e1)
    sweep_ms = sum(a.elapsed_time(b) for a, b in evs)
    total_ms, sweep_ms = replicas.max_over_ranks([total_ms, sweep_ms], dist, sim.device)
    peaks = measured_peaks()
    attempts_per_step = M * L * L
    value = replicas.aggregate_throughput(attempts_per_step, args.steps, world, total_ms)

    # sanity of the state that was timed: sums are consistent with the counters
    S = [int(v) for v in w2_out.cpu().numpy()]
    h00, net = sim.oct_counters()
    assert S[2] == h00 and S[3] == net and S[0] + L * L * h00 == L * L // 2 + 2 * net, "inconsistent state"

    # ---- roofline of the dominant kernel (sweep): issue-slot bound ---------------------------------
    n_sweep_launches = args.steps * M * 4
    launch_s = sweep_ms * 1e-3 / n_sweep_launches
    attempts_per_launch = L * L / 4
    achieved = I_ALG * attempts_per_launch / launch_s / 1e12                     # T lane-instr/s
    peak = N_SM * SMSP * LANES * peaks["sm_max_mhz"] * 1e6 / 1e12
    traffic = None                                   # dram bytes per sweep launch from the committed ncu capture
    tp = os.path.join(ROOT, "profiles", "sweep_traffic.csv")
    if os.path.exists(tp):
        for line in open(tp):
            c = line.strip().split(",")
            if c[0] == f"L{L}_D{1 << args.log2D}" and args.kernel != 1 and args.blk == 0:
                traffic = int(c[1])
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlane-instr/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": "sweep_links_kernel" if (args.log2D <= 7 and args.kernel != 1) else "sweep_kernel", "avg_launch_ms": launch_s * 1e3, "instr_per_attempt": I_ALG,
                "peak_src": f"148 SM x 4 SMSP x 32 lanes x sm_max_mhz ({peaks['src']})",
                "hbm_gbs_of_sweep": 0.5 * (1.0 + 4.0 / (1 << args.log2D)) ** 2 * attempts_per_launch / launch_s / 1e9,
                "sweep_share_of_step": sweep_ms / total_ms}

    # ---- observables (a8/a9): HBM-bound kernels, timed alone, algorithmic bytes / time -------------------
    def time_call(fn, reps=5):
        fn(); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream); torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    lat_bytes = L * L // 4
    observables = {}
    for name, fn, nbytes in (("oct_width2", lambda: sim.oct_width2(w2_out), lat_bytes),
                             ("oct_autocorr", lambda: sim.oct_autocorr(snap, anchor, ac_out), 2 * lat_bytes),
                             ("oct_slope_autocorr", lambda: sim.oct_slope_autocorr(snap, cs_out), 2 * lat_bytes)):
        ms = time_call(fn)
        observables[name] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm": nbytes / ms / 1e6 / peaks["hbm_gbs"]}
    if L <= (1 << 16) and not args.no_heights:
        hbuf = torch.empty((L, L), dtype=torch.int32, device=sim.device)
        ms = time_call(lambda: sim.oct_heights(hbuf), reps=3)
        nbytes = lat_bytes + 4 * L * L
        observables["oct_heights"] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm": nbytes / ms / 1e6 / peaks["hbm_gbs"]}
        del hbuf

    # ---- e2e: same step through the C ABI with HOST buffers ------------------------------------------
    e2e = None
    if not args.no_e2e:
        nb = binding.oct_lattice_bytes(L)
        host = torch.empty(nb // 4, dtype=torch.int32).pin_memory()
        sums_host = torch.empty(9, dtype=torch.int64).pin_memory()
        sim.oct_export_to(host.data_ptr())

        def step_e2e():
            sim.oct_upload(host.data_ptr())
            sim.oct_sweep(M, 1.0, 0.0, code)
            sim.oct_width2(w2_out)
            sim.oct_autocorr(snap, anchor, ac_out)
            sums_host[:4].copy_(w2_out, non_blocking=True)
            sums_host[4:].copy_(ac_out, non_blocking=True)
            sim.oct_export_to(host.data_ptr())                       # synchronises

        ke = max(2, min(args.steps, 5))
        step_e2e()
        barrier()
        t0 = time.perf_counter()
        e0.record(stream)
        for _ in range(ke):
            step_e2e()
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        wall = (time.perf_counter() - t0) * 1e3
        ms = max(ms, wall)
        ms = replicas.max_over_ranks([ms], dist, sim.device)[0]
        e2e = {"value": replicas.aggregate_throughput(attempts_per_step, ke, world, ms), "unit": UNIT, "h2d_bytes_per_step": nb,
               "d2h_bytes_per_step": nb + 72, "steps": ke, "ms_per_step": ms / ke}

    # ---- the oracle timed on this box's host cores (rank 0, N = 1 only) -------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, dt, _ = time_oracle(args.ref_L, min(args.log2D, 8), args.ref_mcs, args.seed)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{args.ref_mcs} MCS of DTrDB(D={1 << args.log2D}) + W2 sums on an L={args.ref_L} flat-start lattice, "
                         f"{dt:.1f} s, oracle/oct_oracle.c gcc -O2 single thread"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
                "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": (value / world / PAPER_ATTEMPTS_PER_S) if (L == 1 << 16) else None,
                "dtype": "u32", "data": "synthetic", "config": workload_config(args), "clocks": clocks, "e2e": e2e,
                "gpu_launches": launches, "roofline": roofline, "observables": observables, "cpu_baseline": cpu,
                "paper_context": "PAPER.md:276 ~9e9 attempts/s on Kepler GPUs (other hardware; context, not a target)"}
        print(json.dumps(line), flush=True)
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
