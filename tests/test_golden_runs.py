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
    assert len(runs) >= 9
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
