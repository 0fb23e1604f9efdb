"""Pins for the oracle's Philox4x32-10 (R19; the paper is silent on the RNG)."""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def _kat():
    rows = []
    with open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = [int(t, 16) for t in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_known_answer_vectors():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert [int(v) for v in oracle.philox4x32_10(ctr, key)] == out


def test_against_curand_host_implementation(tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    so = tmp_path / "libcurand_philox_host.so"
    subprocess.check_call([nvcc, "-O1", "-shared", "-Xcompiler", "-fPIC", "-o", str(so),
                           os.path.join(HERE, "helpers", "curand_philox_host.cu")])
    lib = C.CDLL(str(so))
    lib.curand_philox_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64]
    rng = np.random.default_rng(12345)
    n = 20000
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    # structured counters of the kind the method uses (small c0/c1, tagged c2, small t)
    ctr[: n // 2, 0] %= 64
    ctr[: n // 2, 1] %= 1024
    ctr[: n // 2, 3] %= 10000
    ref = np.zeros((n, 4), dtype=np.uint32)
    lib.curand_philox_host(ctr.ctypes.data, key.ctypes.data, ref.ctypes.data, n)
    for i in range(n):
        assert (oracle.philox4x32_10(ctr[i], key[i]) == ref[i]).all(), i


def test_counter_and_key_sensitivity():
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] ^= 1
        o = oracle.philox4x32_10(c, [5, 6])
        assert (o != base).all()          # every output word depends on every counter word
    for pos in range(2):
        k = [5, 6]
        k[pos] ^= 1
        assert (oracle.philox4x32_10([1, 2, 3, 4], k) != base).all()


def test_words_are_uniform_bits():
    # each of the 32 bit positions of each output word is ~Bernoulli(1/2) over a counter sequence
    n = 4096
    acc = np.zeros((4, 32))
    for i in range(n):
        o = oracle.philox4x32_10([i, 0, 0, 7], [1, 0])
        for w in range(4):
            acc[w] += (int(o[w]) >> np.arange(32)) & 1
    assert np.abs(acc / n - 0.5).max() < 5 * 0.5 / np.sqrt(n)


def test_prob16_thresholds():
    # DESIGN.md R18: P16 = min(65536, floor(p*65536 + 0.5))
    assert oracle.prob16(1.0) == 65536
    assert oracle.prob16(0.0) == 0
    assert oracle.prob16(0.9) == 58982
    assert oracle.prob16(0.1) == 6554
    assert oracle.prob16(0.5) == 32768
