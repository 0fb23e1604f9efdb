"""Stored oracle results (tests/golden/oracle_runs.txt, written by tests/golden/make_oracle_golden.py from oracle/ only).

CPU: the oracle still reproduces them -- a regression pin of its arithmetic (R19 keying, scheme loops), so that later
edits of oracle/oct_oracle.c cannot silently change what "bit-exact" means.
GPU: the CUDA path reproduces the same hashes and sums without the oracle in the loop.
"""
import hashlib
import os

import pytest

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_runs.txt")


def golden_runs():
    runs = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        name, L, seed, p, q, code, t, digest, S1, S2, c, net = line.split()
        runs.setdefault((name, int(L), int(seed), float(p), float(q), int(code)), []).append(
            (int(t), digest, (int(S1), int(S2), int(c), int(net))))
    return runs


def sha(words):
    return hashlib.sha256(words.astype("<u4").tobytes()).hexdigest()


def test_oracle_reproduces_its_golden_runs():
    from oracle import Oracle
    runs = golden_runs()
    assert len(runs) >= 12 and sum(1 for k in runs if k[2] >> 32) >= 3       # three runs with a live high half of the seed
    for (name, L, seed, p, q, code), cps in runs.items():
        o = Oracle(L, seed)
        for t, digest, sums in cps:
            o.sweep(t - o.t, p, q, code)
            assert sha(o.lattice) == digest and o.sums() == sums, (name, t)
        o.close()


@pytest.mark.gpu
def test_gpu_reproduces_the_golden_runs():
    pytest.importorskip("torch")
    from paper_1705_01022_b200 import binding
    for (name, L, seed, p, q, code), cps in golden_runs().items():
        for kernel in (binding.OCT_KERNEL_AUTO, binding.OCT_KERNEL_BITPACKED):
            sim = binding.Sim(L, seed)
            sim.oct_set_option(binding.OCT_OPT_KERNEL, kernel)
            for t, digest, sums in cps:
                sim.oct_sweep(t - sim.oct_mcs(), p, q, code)
                assert sha(sim.oct_export()) == digest, (name, t, kernel)
                assert tuple(int(v) for v in sim.oct_width2().cpu().numpy()) == sums, (name, t, kernel)
            sim.close()


def test_full_size_golden_files_are_complete():
    """The full-size oracle results (make_oracle_golden.py --full) that tests/test_gpu_fullsize.py compares with: every
    run is present with all its checkpoints, and config 4's two domain sizes differ (the hashes pin a scheme, not a size)."""
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    want = {"c4_D64": [1, 2], "c4_D128": [1, 2], "c4_D256": [1, 2], "c4_D64_TC22": [1, 2], "c5_D64": [1],
            "c3_D128": list(range(500, 5001, 500)), "c3_D64": list(range(500, 5001, 500))}
    seen = {}
    for name, ts in want.items():
        rows = [l.split() for l in open(os.path.join(here, f"full_{name}.txt")) if l.strip() and not l.startswith("#")]
        cps = [r for r in rows if r[0] == name]
        assert [int(r[6]) for r in cps] == ts, name
        for r in cps:
            L, S1, net = int(r[1]), int(r[8]), int(r[11])
            assert len(r[7]) == 64 and S1 + L * L * int(r[10]) == L * L // 2 + 2 * net, (name, r[6])   # sum of heights
            seen[(name, r[6])] = r[7]
        if name == "c3_D128":
            assert len([r for r in rows if r[0] == "sums_sha"]) == len(ts)
    assert len(set(seen.values())) == len(seen)
