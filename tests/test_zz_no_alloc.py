"""oct_width2_static: the roughness sums for callers that cannot allocate device memory.

Every other call of liboct_b200 needs a handle, and a handle needs a workspace that the caller allocated.  Some callers
cannot do that: a measurement hook that is given only a lattice pointer and a result slot by a program that owns all of
the GPU's memory, code that must not call cudaMalloc / cudaFree because those stall every stream of the device (other
replicas are sweeping on them), code inside a section of the host program where allocation is forbidden.  For them
`oct_width2_static` keeps its scratch in a fixed array inside the library (L <= 2^16) and allocates nothing.

What is checked here: that it gives exactly the integers of the existing path (`oct_width2` on a handle; the tests of
this repository compare integer sums for equality, there is no tolerance to apply) on two calls in a row -- the second
on a smaller lattice, so that it runs on top of what the first left in the shared scratch, and into an output buffer
that still holds the first result -- and that a lattice beyond the limit is refused with its own error code.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here must not hide other tests).
It needs nothing from the tests before it and leaves nothing behind: it passes alone in a fresh process and at the
end of the whole run.
"""
import ctypes as C

import pytest

from paper_1705_01022_b200 import binding, workloads as wl


def _tuple(t):
    return tuple(int(v) for v in t.cpu().numpy())


@pytest.mark.gpu
def test_static_scratch_width2_equals_the_handle_path_twice_in_a_row():
    import torch
    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    code = wl.scheme_code(wl.DEV_DTR, wl.BLK_DB, 6)
    out = torch.full((4,), -12345, dtype=torch.int64, device=dev)      # reused by both calls, never cleared by the test

    # call 1: L = 2048 (the 16-words-per-lane reduction, 2 CTAs of column words), after a few sweeps with both rates
    big = binding.Sim(2048, 0x9E3779B97F4A7C15, wl.INIT_FLAT, device="cuda:0")
    big.oct_sweep(6, 0.9, 0.1, code)
    want_big = _tuple(big.oct_width2())
    h00, net = big.oct_counters()
    got_big = _tuple(binding.oct_width2_static(big.lattice, 2048, h00, net, out))
    assert got_big == want_big
    assert want_big[2:] == (h00, net)

    # call 2, straight after: L = 256 (the short-row reduction), on the scratch and the output the first call used
    small = binding.Sim(256, 77, wl.INIT_FLAT, device="cuda:0")
    small.oct_sweep(9, 1.0, 0.0, code)
    want_small = _tuple(small.oct_width2())
    h00s, nets = small.oct_counters()
    got_small = _tuple(binding.oct_width2_static(small.lattice, 256, h00s, nets, out))
    assert got_small == want_small
    assert got_small != got_big

    # and the first lattice again: the same integers as before (nothing of call 2 leaks into call 3)
    assert _tuple(binding.oct_width2_static(big.lattice, 2048, h00, net, out)) == want_big

    # a value fixed by the model, not by either path: the flat start has W^2 = 1/4 (S1 = S2 = N/2 with c = 0)
    flat = binding.Sim(1024, 1, wl.INIT_FLAT, device="cuda:0")
    n = 1024 * 1024
    assert _tuple(binding.oct_width2_static(flat.lattice, 1024, 0, 0, out)) == (n // 2, n // 2, 0, 0)
    for s in (big, small, flat):
        s.close()


@pytest.mark.gpu
def test_static_scratch_limit_is_enforced_on_the_gpu_box():
    import torch
    dev = torch.device("cuda:0")
    lat = torch.zeros(64, dtype=torch.int32, device=dev)               # never read: the size check comes first
    out = torch.full((4,), 7, dtype=torch.int64, device=dev)
    with pytest.raises(binding.OctError) as e:
        binding.oct_width2_static(lat, 1 << 17, 0, 0, out)
    assert e.value.code == binding.OCT_ETOOBIG and "65536" in str(e.value)
    torch.cuda.synchronize()
    assert _tuple(out) == (7, 7, 7, 7)                                  # nothing was enqueued


def test_static_scratch_argument_checks_need_no_gpu():
    """The size and pointer checks come before the first CUDA call, so they can be exercised on the CPU box."""
    lib = binding.load()
    fake = 4096                                                         # non-null, aligned; never dereferenced
    assert binding.OCT_WIDTH2_STATIC_MAX_L == 1 << 16
    assert lib.oct_width2_static(fake, 1 << 17, 0, 0, fake, None) == binding.OCT_ETOOBIG
    assert b"oct_width2_static" in lib.oct_strerror(binding.OCT_ETOOBIG) and b"65536" in lib.oct_strerror(binding.OCT_ETOOBIG)
    for bad_L in (0, 8, 100, 3 << 10, 1 << 18):
        assert lib.oct_width2_static(fake, bad_L, 0, 0, fake, None) == binding.OCT_EINVAL
    assert lib.oct_width2_static(None, 256, 0, 0, fake, None) == binding.OCT_EINVAL
    assert lib.oct_width2_static(fake, 256, 0, 0, None, None) == binding.OCT_EINVAL
    assert lib.oct_width2_static(fake + 4, 256, 0, 0, fake, None) == binding.OCT_EINVAL      # lattice not 16-byte aligned
    assert lib.oct_width2_static(fake, 256, 0, 0, fake + 4, None) == binding.OCT_EINVAL      # output not 8-byte aligned
    assert isinstance(lib.oct_width2_static, C._CFuncPtr)
