"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol declared in
include/oct.h, and its pure host helpers / argument checks behave (no compute call needs a GPU)."""
import ctypes as C
import os
import re
from fractions import Fraction

import pytest

from paper_1705_01022_b200 import binding, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "oct.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(oct_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = binding.load()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_sizes_and_L_validation():
    assert binding.oct_lattice_bytes(256) == 256 * 256 // 4
    assert binding.oct_lattice_bytes(1 << 17) == 1 << 32
    assert binding.oct_workspace_bytes(256) == 1280 + 10 * 256
    for bad in (0, 8, 100, 3 << 10, 1 << 18):
        assert binding.oct_lattice_bytes(bad) == 0 and binding.oct_workspace_bytes(bad) == 0


def test_scheme_checks_match_the_header():
    ok = binding.oct_scheme_supported
    for cfg in wl.CONFIGS:
        assert ok(cfg.L, cfg.scheme), cfg.name
    for code in wl.ALL_SCHEMES(5):
        assert ok(128, code)
    assert not ok(128, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 7))            # L < 2D: no room for a 2D x 2D tile
    # the dead-border layers tile with D x D: a single tile (L = D) is valid there, as in the oracle
    import oracle
    for dev in (wl.DEV_DTR, wl.DEV_DT, wl.DEV_DB, wl.DEV_CDB, wl.DEV_DBH):
        for L, lD in ((64, 6), (128, 6), (32, 5), (128, 7), (256, 8), (64, 7)):
            code = wl.scheme_code(dev, wl.BLK_DB, lD)
            assert ok(L, code) == (oracle.lib().orc_check_scheme(L, code) == 0), (dev, L, lD)
    assert ok(64, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6)) and not ok(64, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6))
    assert not ok(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DT, 6, 0, 0))      # DT needs TC >= 1,1 (:182)
    assert not ok(256, wl.scheme_code(5, 0, 6)) and not ok(256, wl.scheme_code(0, 4, 6))
    assert ok(256, wl.scheme_code(wl.DEV_DBH, wl.BLK_DB, 6))
    assert ok(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 6)) and not ok(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DTR, 6, 0, 1))
    assert not ok(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 4))            # D=16 not built
    assert not ok(100, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 5))
    assert not ok(256, -1)


def test_null_and_invalid_arguments_do_not_crash():
    lib = binding.load()
    h = C.c_void_p()
    assert lib.oct_create(None, 256, 1, 0, None, None, None) == binding.OCT_EINVAL
    assert lib.oct_create(C.byref(h), 100, 1, 0, 16, 16, None) == binding.OCT_EINVAL
    assert lib.oct_create(C.byref(h), 256, 1, 0, None, None, None) == binding.OCT_EINVAL
    assert lib.oct_create(C.byref(h), 256, 1, 7, 16, 16, None) == binding.OCT_EINVAL
    assert lib.oct_sweep(None, 1, 1.0, 0.0, 0, None) == binding.OCT_EINVAL
    assert lib.oct_sweep_batch(None, 1, 1, 1.0, 0.0, 0, None) == binding.OCT_EINVAL
    two = (C.c_void_p * 2)(None, None)
    assert lib.oct_sweep_batch(two, 2, 1, 1.0, 0.0, 0, None) == binding.OCT_EINVAL
    assert lib.oct_sweep_batch(two, 0, 1, 1.0, 0.0, 0, None) == binding.OCT_EINVAL
    assert lib.oct_destroy(None) == binding.OCT_EINVAL
    assert lib.oct_strerror(0) == b"ok" and lib.oct_strerror(-1) == b"invalid argument"
    assert lib.oct_last_error(None) == b""


def test_host_helpers_are_exact_rationals_rounded_once():
    L = 1 << 16
    N = L * L
    S1, S2 = 123456789012345, 98765432109876543
    exact = Fraction(N * S2 - S1 * S1, N * N)
    assert binding.oct_w2_from_sums(L, S1, S2) == pytest.approx(float(exact), rel=1e-15)
    St, Ss, Sts = -5_000_000_007, 9_000_000_011, 77_777_777_777_777
    exact = Fraction(N * Sts - St * Ss, N * N)
    assert binding.oct_c_from_sums(L, St, Ss, Sts) == pytest.approx(float(exact), rel=1e-15)
    assert binding.oct_w2_from_sums(256, 256 * 256 // 2, 256 * 256 // 2) == 0.25       # flat start (R5)


def test_t_async_and_width_fields():
    ok = binding.oct_scheme_supported
    import oracle
    for dev in (wl.DEV_DTR, wl.DEV_DT, wl.DEV_DB, wl.DEV_CDB, wl.DEV_DBH):
        for ka in (0, 1, 2, 3):
            for w in (0, 1, 5, 7):
                for tc in (0, 1):
                    code = wl.scheme_code(dev, wl.BLK_DB, 6, tc, tc, ka, w)
                    assert ok(256, code) == (oracle.lib().orc_check_scheme(256, code) == 0), (dev, ka, w, tc)
    assert ok(256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 2, 1)) and not ok(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6, 1, 1, 1, 0))
    assert not ok(256, 1 << 26)
    assert binding.oct_time_per_sweep(256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6, 1, 1, 2, 1)) == pytest.approx((63 / 64) ** 2)
    assert binding.oct_time_per_sweep(256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DB, 6, 1, 1, 0, 3)) == pytest.approx((61 / 64) ** 2)


def test_time_per_sweep_eq9():
    # Eq. (9) with reading R9: a DB sweep lasts (N - N_border)/N MCS
    assert binding.oct_time_per_sweep(256, wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)) == 1.0
    assert binding.oct_time_per_sweep(256, wl.scheme_code(wl.DEV_DB, wl.BLK_DB, 6)) == pytest.approx((59 / 64) ** 2)
    assert binding.oct_time_per_sweep(256, wl.scheme_code(wl.DEV_CDB, wl.BLK_DB, 6)) == pytest.approx((63 / 64) ** 2)


def test_no_gpu_means_loud_failure_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU box")
    with pytest.raises(binding.OctError):
        binding.Sim(256, 1)
