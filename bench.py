#!/usr/bin/env python
"""bench.py -- throughput of the DD random-sequential sweep of the octahedron model on B200.

    python bench.py --gpus N --steps K --warmup W            (N>1: launched by torch.distributed.run)
    python bench.py --impl reference ...                     (times the CPU oracle instead)

Metric (BASELINE.json): site-update attempts per second at L = 2^16, p = 1, q = 0, scheme DTrDB
(PAPER.md:262, :276).  One *step* is one pass of the whole hot path on the resident lattice:
`--mcs-per-step` MCS of oct_sweep (4 launches per MCS), then the W^2 and C_h sums against the waiting-time
snapshot in one pass (oct_observe).  attempts = mcs_per_step * L^2 per step (rejected attempts count, :270).
The lattice (1 GiB) is larger than L2 (126 MB), so no explicit L2 flush is needed between steps.
The same run also measures L = 2^17 (`also`), the second size BASELINE.json's north_star names.
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

# the paper's DTrDB throughput at L = 2^16, p=1, q=0 on Kepler GPUs, per GPU
PAPER_ATTEMPTS_PER_S = 9.0e9
N_SM, SMSP, LANES = 148, 4, 32
# Conflict-free minimum of shared-memory wavefronts per warp-attempt (32 update attempts) of the link-entry sweep
# (DESIGN.md section 5.1).  Four-byte entries: 1 entry load + 5 stores of an accepted update (issued whenever a lane of the
# warp accepts); two-byte entries (shapes with few cells per domain): 3 loads + 3 stores.  Plus staging in and out,
# 2 x ((D+4)^2 entries x EB bytes / 128 B) per D^2/32 warp-attempts of a domain, plus 1/8 block-step load.
TWO_BYTE_SHAPES = {(6, 2, 2), (7, 2, 2), (7, 3, 2), (7, 4, 1), (8, 1, 1), (8, 2, 1), (8, 2, 2)}   # (log2D, tcx, tcy), as built in csrc/sweep_inst.cu


def wavefronts_min(log2D: int, tcx: int, tcy: int, kernel_opt: int = 0) -> float:
    eb = 2 if ((log2D, tcx, tcy) in TWO_BYTE_SHAPES and kernel_opt != 2) else 4
    D = 1 << log2D
    staging = 2.0 * ((D + 4) * (D + 4) * eb / 128.0) / (D * D / 32.0)
    return 6.0 + staging + 0.125          # six loads and stores per attempt in either layout (1 + 5 or 3 + 3)


WAVEFRONTS_MIN = wavefronts_min(6, 1, 1)


def expected_max_bank_load(n_lanes, n_banks=32, trials=20000, seed=12345):
    """E[max number of lanes that fall into one bank] for n_lanes accesses at independent uniformly random banks: the
    wavefronts one shared-memory instruction costs when its lanes address unrelated 32-bit words.
    n_lanes may be an array of per-trial lane counts (stores: only the accepting lanes are live)."""
    import numpy as np
    rng = np.random.default_rng(seed)
    n = np.broadcast_to(np.asarray(n_lanes), (trials,))
    banks = rng.integers(0, n_banks, size=(trials, 32))
    live = np.arange(32)[None, :] < n[:, None]
    occ = np.zeros((trials, n_banks), dtype=np.int64)
    np.add.at(occ, (np.repeat(np.arange(trials), 32)[live.ravel()], banks.ravel()[live.ravel()]), 1)
    return float(occ.max(axis=1).mean())


def wavefronts_expected_linear(log2D, tcx, tcy, kernel_opt, acceptance, trials=20000):
    """Expected shared-memory wavefronts per warp-attempt of the link-entry sweep in ANY layout that is linear in the site
    coordinates (entry address = y * pitch + x): the 32 lanes of a collective step address 32 unrelated sites, so every
    load costs E[max bank load of 32 random banks] ~ 3.5 wavefronts instead of 1, and every store instruction -- issued
    for the warp whenever a lane accepts, with only the accepting lanes live -- E[max(1, max bank load of n)] with
    n ~ Binomial(32, acceptance).  Staging and the block-step load stay conflict-free.  This is the ceiling of the layout,
    not of the hardware: roofline.frac is quoted against the conflict-free minimum, frac_of_layout_ceiling against this."""
    import numpy as np
    eb = 2 if ((log2D, tcx, tcy) in TWO_BYTE_SHAPES and kernel_opt != 2) else 4
    n_loads, n_stores = (1, 5) if eb == 4 else (3, 3)
    rng = np.random.default_rng(777)
    load = expected_max_bank_load(32, trials=trials)
    n_acc = rng.binomial(32, acceptance, size=trials)
    store = expected_max_bank_load(np.maximum(n_acc, 1), trials=trials)
    conflict_free_rest = wavefronts_min(log2D, tcx, tcy, kernel_opt) - 6.0
    return {"wavefronts_expected_linear": n_loads * load + n_stores * store + conflict_free_rest, "per_load": load, "per_store": store,
            "acceptance": acceptance, "loads": n_loads, "stores": n_stores,
            "model": "lanes at independent uniformly random banks (32 banks x 4 B); stores with Binomial(32, acceptance) live lanes"}
# Algorithmic lane-instructions per attempt: Philox 40/4 = 10, site select 5, entry load +
# compare 2, five stores + accept count 6, loop/sync 1, staging per site 6 (permute expansion 47/16, gather 34/16, loads,
# stores and addresses).  The executed count comes from the committed ncu capture.
I_ALG = 30.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": d.get("hbm_gbs", 6650.0), "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


def ncu_counters(kernel: str, L: int, log2D: int, tcx: int, tcy: int, blk: int, p: float = 1.0, q: float = 0.0):
    """Per-launch counters of the sweep kernel from the committed ncu capture (profiles/sweep_counters.csv: one row per
    captured configuration; the .md beside it names the command).  None if this configuration was not captured."""
    path = os.path.join(ROOT, "profiles", "sweep_counters.csv")
    if not os.path.exists(path):
        return None
    rows = [l.strip().split(",") for l in open(path) if l.strip() and not l.startswith("#")]
    hdr = rows[0]
    for r in rows[1:]:
        d = dict(zip(hdr, r))
        if (d["kernel"], int(d["L"]), int(d["log2D"]), int(d["tcx"]), int(d["tcy"]), int(d["blk"]), float(d.get("p", 1.0)), float(d.get("q", 0.0))) == \
                (kernel, L, log2D, tcx, tcy, blk, float(p), float(q)):
            return {k: (float(v) if k not in ("kernel", "source") else v) for k, v in d.items()}
    return None


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


def scheme_label(args):
    name = "DTrDT" if getattr(args, "blk", 0) == 2 else "DTrDB"
    return f"{name},TC={args.tcx},{args.tcy},D={1 << args.log2D}"


def baseline_config_no(L):
    return {256: 1, 1024: 2, 4096: 3, 1 << 16: 4, 1 << 17: 5}.get(L)


def workload_config(args, oracle_sample_L=None):
    n = baseline_config_no(args.L)
    tag = f"BASELINE config {n}" if n else "custom size"
    pp, qq = getattr(args, "p", 1.0), getattr(args, "q", 0.0)
    if (pp, qq) != (1.0, 0.0):
        tag = "custom rates"
    cfg = {"workload": f"{tag}: octahedron model, L={args.L} periodic, flat start, p={pp:g} q={qq:g}, {scheme_label(args)}",
           "L": args.L, "p": pp, "q": qq, "scheme": scheme_label(args), "mcs_per_step": args.mcs_per_step,
           "burn_in_mcs": args.burn_in, "l2": "inputs larger than L2 (lattice %d MiB)" % (args.L * args.L // 4 >> 20),
           "parallelism": f"replicas x{args.gpus}" if args.gpus > 1 else "single GPU"}
    if oracle_sample_L is not None:
        cfg["timed_sample"] = f"the oracle is timed on an L={oracle_sample_L} sample of this workload (same scheme, p, q, domain size)"
        cfg["sample_L"] = oracle_sample_L
    return cfg


def time_oracle(L: int, code_args, n_mcs: int, seed: int, burn: int = 1, rs: bool = False):
    """The CPU oracle as it stands, single thread, on a bounded sample of the workload (attempts/s, seconds, sums)."""
    import oracle
    log2D, tcx, tcy, blk = code_args
    code = oracle.scheme(oracle.DEV_DTR, blk, log2D, tcx, tcy)
    o = oracle.Oracle(L, seed)
    run = (lambda n: o.sweep_rs(n, 1.0, 0.0)) if rs else (lambda n: o.sweep(n, 1.0, 0.0, code))
    run(burn)                                # leave the exactly-flat state (acceptance 0.5 -> ~0.2)
    t0 = time.perf_counter()
    run(n_mcs)
    S = o.sums(rowpath=True)
    dt = time.perf_counter() - t0
    o.close()
    return n_mcs * L * L / dt, dt, S


def run_reference(args, rank: int, world: int):
    if rank != 0:
        return
    Ls, n_mcs = args.ref_L, args.ref_mcs
    ca = (min(args.log2D, 8), args.tcx, args.tcy, args.blk)
    vals, times = [], []
    for i in range(args.warmup + args.steps):
        v, dt, _ = time_oracle(Ls, ca, n_mcs, args.seed + i, burn=args.ref_burn)
        if i >= args.warmup:
            vals.append(v); times.append(dt)
    value = sum(vals) / len(vals)
    sample = (f"per step: {n_mcs} MCS of {scheme_label(args)} incl. the W2 sums on an L={Ls} lattice after {args.ref_burn} burn-in MCS from flat "
              f"(same scheme, p, q and domain size as the L={args.L} workload; oracle/oct_oracle.c, gcc -O2, 1 thread)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": workload_config(args, oracle_sample_L=Ls),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def measure(sim, code, M, steps, warmup, torch, dist, replicas, binding, snap, anchor, obs_out, sampler=None, p=1.0, q=0.0):
    """warmup + `steps` timed steps of (M MCS of oct_sweep, then W^2 and C_h sums in one pass); CUDA events on the stream."""
    stream = torch.cuda.current_stream()
    what = binding.OCT_OBS_W2 | binding.OCT_OBS_CH

    def step(ev=None):
        if ev:
            ev[0].record(stream)
        sim.oct_sweep(M, p, q, code)
        if ev:
            ev[1].record(stream)
        sim.oct_observe(what, snap, anchor, obs_out)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    barrier()
    if sampler is not None:
        sampler.start()
    n0 = sim.oct_launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(steps):
        step(evs[i])
    e1.record(stream)
    barrier()
    launches = sim.oct_launch_count() - n0
    clocks = sampler.stop() if sampler is not None else None
    total_ms = e0.elapsed_time(e1)
    per_step_sweep = [a.elapsed_time(b) for a, b in evs]
    total_ms, sweep_ms = replicas.max_over_ranks([total_ms, sum(per_step_sweep)], dist, sim.device)
    return {"total_ms": total_ms, "sweep_ms": sweep_ms, "launches": launches, "clocks": clocks, "barrier": barrier,
            "window_ms": per_step_sweep}


def roofline_block(args, L, peaks, sweep_ms, total_ms, n_sweep_launches, kernel, acceptance=None):
    """Roofline of the dominant kernel (one domain-set sweep): shared-memory data pipe, with the issue-slot view beside it."""
    launch_s = sweep_ms * 1e-3 / n_sweep_launches
    attempts_per_launch = L * L / 4
    warp_attempts = attempts_per_launch / 32
    f_hz = peaks["sm_max_mhz"] * 1e6
    peak_wf = N_SM * f_hz / 1e9                                    # G wavefronts/s: one per clock per SM
    wf_min = wavefronts_min(args.log2D, args.tcx, args.tcy, args.kernel)
    achieved = wf_min * warp_attempts / launch_s / 1e9
    pq = (getattr(args, "p", 1.0), getattr(args, "q", 0.0))
    cnt = ncu_counters(kernel, L, args.log2D, args.tcx, args.tcy, args.blk, *pq) or ncu_counters(kernel, 1 << 16, args.log2D, args.tcx, args.tcy, args.blk, *pq)
    rf = {"bound": "smem", "achieved": achieved, "peak": peak_wf, "unit": "Gwavefront/s", "frac": achieved / peak_wf,
          "traffic": None, "kernel": kernel, "avg_launch_ms": launch_s * 1e3, "attempts_per_launch": attempts_per_launch,
          "wavefronts_per_warp_attempt_min": wf_min,
          "peak_src": f"148 SM x 1 shared-memory wavefront/clk x sm_max_mhz ({peaks['src']})",
          "hbm_gbs_of_sweep": 0.5 * (1.0 + 4.0 / (1 << args.log2D)) ** 2 * attempts_per_launch / launch_s / 1e9,
          "sweep_share_of_step": sweep_ms / total_ms}
    peak_issue = N_SM * SMSP * LANES * f_hz / 1e12
    issue = {"unit": "Tlane-instr/s", "peak": peak_issue, "instr_per_attempt_algorithmic": I_ALG,
             "achieved_algorithmic": I_ALG * attempts_per_launch / launch_s / 1e12}
    issue["frac_algorithmic"] = issue["achieved_algorithmic"] / peak_issue
    if cnt is not None:
        scale = attempts_per_launch / (cnt["L"] * cnt["L"] / 4)        # counters of an L = 2^16 capture scale with the domain count
        rf["traffic"] = int(cnt["dram_bytes"] * scale)
        wpa = cnt["wavefronts_shared"] / (cnt["L"] * cnt["L"] / 4 / 32)
        rf["wavefronts_per_warp_attempt_measured"] = wpa
        rf["pipe_utilisation"] = wpa * warp_attempts / launch_s / 1e9 / peak_wf
        ipa = cnt["inst_executed"] / (cnt["L"] * cnt["L"] / 4 / 32)
        issue["instr_per_attempt_executed"] = ipa
        issue["achieved_executed"] = ipa * attempts_per_launch / launch_s / 1e12
        issue["frac_executed"] = issue["achieved_executed"] / peak_issue
        rf["counters_src"] = cnt["source"]
    rf["issue_slots"] = issue
    if acceptance is not None and kernel == "sweep_links_kernel":
        lc = wavefronts_expected_linear(args.log2D, args.tcx, args.tcy, args.kernel, acceptance)
        lc["frac_of_layout_ceiling"] = lc["wavefronts_expected_linear"] * warp_attempts / launch_s / 1e9 / peak_wf
        rf["layout_ceiling"] = lc
    return rf


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--L", type=int, default=1 << 16)
    ap.add_argument("--log2D", type=int, default=6)
    ap.add_argument("--mcs-per-step", type=int, default=32)
    ap.add_argument("--burn-in", type=int, default=32)
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--p", type=float, default=1.0, help="deposition probability of the timed workload (BASELINE config 4: 1)")
    ap.add_argument("--q", type=float, default=0.0, help="removal probability (config 4: 0; config 3's mixed rates: --p 0.9 --q 0.1)")
    ap.add_argument("--ref-L", type=int, default=4096, help="lattice edge of the oracle's timed sample")
    ap.add_argument("--ref-mcs", type=int, default=16)
    ap.add_argument("--ref-burn", type=int, default=4)
    ap.add_argument("--tcx", type=int, default=1, help="thread-cell size TC=tcx,tcy (log2 of the cell edge in 4-site words, PAPER.md:180)")
    ap.add_argument("--tcy", type=int, default=1)
    ap.add_argument("--blk", type=int, default=0, help="block layer: 0 DB (the benched DTrDB), 2 DT (DTrDT, PAPER.md:268)")
    ap.add_argument("--kernel", type=int, default=0, help="OCT_OPT_KERNEL value: 0 auto, 1 bit-packed, 2 link-entry variant B")
    ap.add_argument("--also-L", type=int, default=1 << 17, help="second lattice size measured in the same run (0: none)")
    ap.add_argument("--ensemble-L", type=int, default=1024, help="lattice edge of the ensemble (many lattices per launch) measurement (0: none)")
    ap.add_argument("--no-shapes", dest="shapes", action="store_false", help="skip the other-shapes block")
    ap.add_argument("--shapes-all", action="store_true", help="the other-shapes block over every Fig. 4 cell shape x D x kernel option x rate set (minutes)")
    ap.add_argument("--sustained-windows", type=int, default=3, help="windows of the sustained-throughput protocol (0: skip)")
    ap.add_argument("--sustained-window-mcs", type=int, default=100, help="MCS per window (at least 100)")
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

    if rank == 0:                                # one rank builds (if stale) before the others load the library
        from paper_1705_01022_b200 import binding
        binding.load()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    from paper_1705_01022_b200 import binding, replicas, workloads as wl

    L, M = args.L, args.mcs_per_step
    code = wl.scheme_code(wl.DEV_DTR, args.blk, args.log2D, args.tcx, args.tcy)
    seed = replicas.replica_seed(args.seed, rank)
    warm = max(args.warmup, 3)
    peaks = measured_peaks()
    links_shape = args.log2D <= 7 or (args.log2D == 8 and (args.tcx, args.tcy) in ((1, 1), (2, 1), (2, 2)))
    kernel = "sweep_links_kernel" if (links_shape and args.kernel != 1) else "sweep_kernel"

    sim = binding.Sim(L, seed, wl.INIT_FLAT, device=f"cuda:{local_rank}")
    sim.oct_set_option(binding.OCT_OPT_KERNEL, args.kernel)
    stream = torch.cuda.current_stream()
    sim.oct_sweep(args.burn_in, args.p, args.q, code)      # evolved state: acceptance ~0.2 (not the flat 0.5)
    snap, anchor = sim.oct_snapshot()
    obs = torch.empty(16, dtype=torch.int64, device=sim.device)
    net_before = sim.oct_counters()[1]
    m = measure(sim, code, M, args.steps, warm, torch, dist, replicas, binding, snap, anchor, obs,
                sampler=ClockSampler(local_rank) if rank == 0 else None, p=args.p, q=args.q)
    # acceptance over warm-up + timed steps: with one rate zero every accepted update moves the net counter by one
    # (mixed rates: deposits and removals cancel in it, so no figure and no layout ceiling there)
    acceptance = None
    if args.p == 0.0 or args.q == 0.0:
        acceptance = abs(sim.oct_counters()[1] - net_before) / float((warm + args.steps) * M * L * L)
    barrier = m["barrier"]
    attempts_per_step = M * L * L
    value = replicas.aggregate_throughput(attempts_per_step, args.steps, world, m["total_ms"])

    # sanity of the state that was timed: sums are consistent with the counters
    S = [int(v) for v in obs.cpu().numpy()]
    h00, net = sim.oct_counters()
    assert S[2] == h00 and S[3] == net and S[0] + L * L * h00 == L * L // 2 + 2 * net and S[4] == S[0], "inconsistent state"

    roofline = roofline_block(args, L, peaks, m["sweep_ms"], m["total_ms"], args.steps * M * 4, kernel, acceptance)
    # Sustained throughput, the protocol of SURVEY 8(d): the paper saw its GPU clock down after ~100 MCS (PAPER.md:262, :268,
    # Fig. 7), so the figure is the MEDIAN over windows of >= 100 MCS that start after >= 200 MCS of load.  Everything
    # above (burn-in, warm-up, the timed steps) is that load; the windows are sweeps only, timed with CUDA events, with the
    # clock sampler running.
    sustained = None
    if args.sustained_windows > 0:
        mcs_before = args.burn_in + (warm + args.steps) * M
        extra = max(0, 200 - mcs_before)
        if extra:
            sim.oct_sweep(extra, args.p, args.q, code)
        Wm = max(100, args.sustained_window_mcs)
        smp = ClockSampler(local_rank) if rank == 0 else None
        evw = [torch.cuda.Event(enable_timing=True) for _ in range(args.sustained_windows + 1)]
        barrier()
        if smp is not None:
            smp.start()
        evw[0].record(stream)
        for i in range(args.sustained_windows):
            sim.oct_sweep(Wm, args.p, args.q, code)
            evw[i + 1].record(stream)
        barrier()
        wclk = smp.stop() if smp is not None else None
        wms = [evw[i].elapsed_time(evw[i + 1]) for i in range(args.sustained_windows)]
        wms = replicas.max_over_ranks(wms, dist, sim.device)
        win = sorted(world * L * L * Wm / (w * 1e-3) for w in wms)
        sustained = {"window_mcs": Wm, "windows": len(win), "mcs_of_load_before_first_window": mcs_before + extra,
                     "median_attempts_per_s": statistics.median(win), "min": win[0], "max": win[-1], "clocks": wclk,
                     "protocol": "median over windows of >= 100 MCS after >= 200 MCS of load (SURVEY 8(d); PAPER.md:262, :268)"}

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
    w2_out = torch.empty(4, dtype=torch.int64, device=sim.device)
    ac_out = torch.empty(5, dtype=torch.int64, device=sim.device)
    cs_out = torch.empty(6, dtype=torch.int64, device=sim.device)
    observables = {}
    for name, fn, nbytes in (("oct_width2", lambda: sim.oct_width2(w2_out), lat_bytes),
                             ("oct_autocorr", lambda: sim.oct_autocorr(snap, anchor, ac_out), 2 * lat_bytes),
                             ("oct_slope_autocorr", lambda: sim.oct_slope_autocorr(snap, cs_out), 2 * lat_bytes),
                             ("oct_observe(W2|CH|CS)", lambda: sim.oct_observe(7, snap, anchor, obs), 2 * lat_bytes)):
        ms = time_call(fn)
        observables[name] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm": nbytes / ms / 1e6 / peaks["hbm_gbs"]}
    if L <= (1 << 16) and not args.no_heights:
        hbuf = torch.empty((L, L), dtype=torch.int32, device=sim.device)
        ms = time_call(lambda: sim.oct_heights(hbuf), reps=3)
        nbytes = lat_bytes + 4 * L * L
        observables["oct_heights"] = {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6, "frac_of_hbm": nbytes / ms / 1e6 / peaks["hbm_gbs"]}
        del hbuf

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned): the lattice goes up before and comes back
    # after the sweeps, the sums come back through oct_fetch -----------------------------------------------
    e2e = None
    if not args.no_e2e:
        nb = binding.oct_lattice_bytes(L)
        host = torch.empty(nb // 4, dtype=torch.int32).pin_memory()
        sums_host = torch.empty(16, dtype=torch.int64).pin_memory()
        sim.oct_export_to(host.data_ptr())
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

        def step_e2e():
            sim.oct_upload(host.data_ptr())                          # the lattice exported by the previous step: counters stay valid
            sim.oct_sweep(M, args.p, args.q, code)
            sim.oct_observe(binding.OCT_OBS_W2 | binding.OCT_OBS_CH, snap, anchor, obs)
            sim.oct_fetch(obs, sums_host.data_ptr(), 16 * 8)         # synchronises
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
        ms = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3)
        ms = replicas.max_over_ranks([ms], dist, sim.device)[0]
        assert int(sums_host[3]) == sim.oct_counters()[1]
        e2e = {"value": replicas.aggregate_throughput(attempts_per_step, ke, world, ms), "unit": UNIT, "h2d_bytes_per_step": nb,
               "d2h_bytes_per_step": nb + 128, "steps": ke, "ms_per_step": ms / ke}
        del host
    sim.close()
    del snap, sim

    # ---- the second size north_star names (L = 2^17: 4 GiB packed), same scheme, in the same run ------------
    also = None
    if args.also_L and args.also_L != L and world == 1:
        L2 = args.also_L
        sim2 = binding.Sim(L2, seed, wl.INIT_FLAT, device=f"cuda:{local_rank}")
        sim2.oct_set_option(binding.OCT_OPT_KERNEL, args.kernel)
        sim2.oct_sweep(args.burn_in, 1.0, 0.0, code)
        snap2, anchor2 = sim2.oct_snapshot()
        M2, K2 = max(1, M // 4), max(3, args.steps // 2)
        m2 = measure(sim2, code, M2, K2, 3, torch, dist, replicas, binding, snap2, anchor2, obs)
        v2 = M2 * L2 * L2 * K2 / (m2["total_ms"] * 1e-3)
        a2 = argparse.Namespace(**vars(args)); a2.L = L2; a2.mcs_per_step = M2
        also = {"config": workload_config(a2), "value": v2, "unit": UNIT, "steps": K2, "ms_per_step": m2["total_ms"] / K2,
                "roofline": roofline_block(args, L2, peaks, m2["sweep_ms"], m2["total_ms"], K2 * M2 * 4, kernel)}
        sim2.close()
        del snap2, sim2

    # ---- ensembles of small lattices, all members in every launch (oct_sweep_batch; the paper's
    # curves are means over n = 20 ... 4367 runs): sweeps only, same scheme ------------------------------------------
    ensemble = None
    if args.ensemble_L and world == 1:
        ensemble = []
        Le = args.ensemble_L
        for n_mem in (1, 32, 256):
            sims = [binding.Sim(Le, seed + 1 + i, wl.INIT_FLAT, device=f"cuda:{local_rank}") for i in range(n_mem)]
            run = (lambda n: binding.oct_sweep_batch(sims, n, 1.0, 0.0, code)) if n_mem > 1 else (lambda n: sims[0].oct_sweep(n, 1.0, 0.0, code))
            run(args.burn_in)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            Me = 200
            a.record(stream); run(Me); b.record(stream); torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            ensemble.append({"L": Le, "members": n_mem, "mcs": Me, "ms": ms, "attempts_per_s": n_mem * Me * Le * Le / (ms * 1e-3),
                             "domains_per_launch": n_mem * (Le >> (args.log2D + 1)) ** 2})
            for sm in sims:
                sm.close()
            del sims

    # ---- other scheme shapes of the same workload (sweeps only, 8 MCS after 16 burn-in MCS): the paper's second production
    # configuration TC=2,2 (Fig. 5 :236-244), larger domains, block-layer DT, and the mixed-rate path of BASELINE config 3 ------
    shapes = None
    if args.shapes and world == 1:
        shapes = []
        shape_list = [(6, 2, 2, 0, 1.0, 0.0, 0), (6, 3, 1, 0, 1.0, 0.0, 0), (7, 1, 1, 0, 1.0, 0.0, 0), (8, 1, 1, 0, 1.0, 0.0, 0), (6, 1, 1, 2, 1.0, 0.0, 0),
                      (6, 1, 1, 0, 0.9, 0.1, 0), (7, 1, 1, 0, 0.9, 0.1, 0)]
        if args.shapes_all:      # every cell shape of the Fig. 4 caption at every D it is built for, both kernels, both rate sets
            shape_list = [(ld, tx, ty, 0, p_, q_, k_) for ld, tx, ty in ((6, 1, 1), (6, 2, 1), (6, 2, 2), (6, 3, 1), (6, 1, 3), (7, 1, 1), (7, 2, 2), (7, 3, 1),
                                                                          (7, 1, 3), (7, 3, 2), (7, 4, 1), (8, 1, 1), (8, 2, 2), (8, 3, 2), (8, 4, 1))
                          for p_, q_ in ((1.0, 0.0), (0.9, 0.1)) for k_ in (0, 1)]
        for log2D, tcx, tcy, blk, p_, q_, k_ in shape_list:
            code_s = wl.scheme_code(wl.DEV_DTR, blk, log2D, tcx, tcy)
            sim_s = binding.Sim(L, seed, wl.INIT_FLAT, device=f"cuda:{local_rank}")
            sim_s.oct_set_option(binding.OCT_OPT_KERNEL, k_)
            sim_s.oct_sweep(16, p_, q_, code_s)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); sim_s.oct_sweep(8, p_, q_, code_s); b.record(stream); torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            shapes.append({"scheme": wl.scheme_name(code_s), "p": p_, "q": q_, "kernel_option": k_, "L": L, "mcs": 8, "launch_ms": ms / 32,
                           "attempts_per_s": 8 * L * L / (ms * 1e-3)})
            sim_s.close()
            del sim_s

    # ---- the oracle timed on this box's host cores (rank 0, N = 1 only): bounded samples ------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ca = (min(args.log2D, 8), args.tcx, args.tcy, args.blk)
        v, dt, _ = time_oracle(args.ref_L, ca, args.ref_mcs, args.seed, burn=args.ref_burn)
        v14, dt14, _ = time_oracle(1 << 14, ca, 2, args.seed, burn=1)
        vrs, dtrs, _ = time_oracle(args.ref_L, ca, 4, args.seed, burn=1, rs=True)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{args.ref_mcs} MCS of {scheme_label(args)} + W2 sums on an L={args.ref_L} lattice ({args.ref_L * args.ref_L // 4 >> 20} MiB, cache-resident: "
                         f"the oracle's most favourable case, cf. the paper's L=2^12 CPU figure, PAPER.md:270) after {args.ref_burn} burn-in MCS, "
                         f"{dt:.1f} s, oracle/oct_oracle.c gcc -O2 single thread; the GPU figure is L={L} after {args.burn_in} burn-in MCS",
               "others": [
                   {"what": f"{scheme_label(args)}, L=16384 (64 MiB, out of cache), 2 MCS after 1", "value": v14, "seconds": dt14},
                   {"what": f"true RS dynamics (PAPER.md:15/:44), L={args.ref_L}, 4 MCS after 1", "value": vrs, "seconds": dtrs}]}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
                "ms_per_step": m["total_ms"] / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None,
                "dtype": "u32", "data": "synthetic", "config": workload_config(args), "clocks": m["clocks"], "e2e": e2e,
                "gpu_launches": m["launches"], "roofline": roofline, "sustained": sustained, "also": also, "ensemble": ensemble, "shapes": shapes,
                "observables": observables, "cpu_baseline": cpu,
                "vs_cpu_baseline": (value / world / cpu["value"]) if cpu else None,
                "paper_context": {"paper_attempts_per_s": PAPER_ATTEMPTS_PER_S,
                                  "value_over_paper": (value / world / PAPER_ATTEMPTS_PER_S) if (L == 1 << 16 and args.blk == 0 and args.p == 1.0 and args.q == 0.0) else None,
                                  "note": "PAPER.md:276: ~9e9 attempts/s for DTrDB at L=2^16, p=1, q=0 on Kepler GPUs -- another machine's number: context, "
                                          "not a baseline (vs_baseline stays null; BASELINE.json publishes none); vs_cpu_baseline divides by the oracle "
                                          "timed in this run (cpu_baseline.sample says on what)"}}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
