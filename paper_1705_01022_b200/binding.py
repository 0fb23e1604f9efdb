"""ctypes binding of liboct_b200.so -- argument marshalling only.

Every function below has the name and the arguments of its C declaration in ``include/oct.h``; device
buffers are ``torch`` CUDA tensors (PyTorch is used for device memory and streams only) and are passed
as raw pointers.  ``Sim`` bundles a handle with the buffers it lives on.  There is no fallback of any
kind: if the library cannot be loaded, or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build
from . import workloads as wl

OCT_OK, OCT_EINVAL, OCT_ECUDA, OCT_ENOMEM, OCT_ESTATE = 0, -1, -2, -3, -4
OCT_ETOOBIG = -5
OCT_WIDTH2_STATIC_MAX_L = 1 << 16

EXPORTS = (
    "oct_lattice_bytes", "oct_workspace_bytes", "oct_create", "oct_set_state", "oct_sweep", "oct_heights",
    "oct_width2", "oct_snapshot", "oct_autocorr", "oct_export", "oct_upload", "oct_counters", "oct_mcs",
    "oct_destroy", "oct_strerror", "oct_last_error", "oct_launch_count", "oct_w2_from_sums", "oct_c_from_sums",
    "oct_time_per_sweep", "oct_scheme_supported", "oct_set_option", "oct_slope_autocorr", "oct_cs_from_sums",
    "oct_sweep_batch", "oct_observe", "oct_fetch", "oct_observe_batch", "oct_width2_static",
)
OCT_OBS_W2, OCT_OBS_CH, OCT_OBS_CS = 1, 2, 4
OCT_OPT_KERNEL = 1
OCT_KERNEL_AUTO, OCT_KERNEL_BITPACKED, OCT_KERNEL_LINKS_B = 0, 1, 2


class OctError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where} -> {code} ({_strerror(code)}){': ' + detail if detail else ''}")


_lib = None


def lib_path() -> str:
    return _build.LIB


def load(rebuild_if_stale: bool = True):
    """Load the product library; build it first when sources are newer and nvcc exists."""
    global _lib
    if _lib is not None:
        return _lib
    if rebuild_if_stale and _build.stale():
        _build.build()
    if not os.path.exists(_build.LIB):
        raise ImportError(f"{_build.LIB} is missing: run `python -m paper_1705_01022_b200.build` (needs nvcc)")
    L = C.CDLL(_build.LIB)
    vp, u32, u64, i64, i32, dbl, sz = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int64, C.c_int, C.c_double, C.c_size_t
    sig = {
        "oct_lattice_bytes": (sz, [u32]), "oct_workspace_bytes": (sz, [u32]),
        "oct_create": (i32, [C.POINTER(vp), u32, u64, i32, vp, vp, vp]),
        "oct_set_state": (i32, [vp, u64, i64, i64, vp]),
        "oct_sweep": (i32, [vp, u64, dbl, dbl, i32, vp]),
        "oct_sweep_batch": (i32, [C.POINTER(vp), u32, u64, dbl, dbl, i32, vp]),
        "oct_heights": (i32, [vp, vp, vp]), "oct_width2": (i32, [vp, vp, vp]),
        "oct_snapshot": (i32, [vp, vp, vp, vp]), "oct_autocorr": (i32, [vp, vp, vp, vp, vp]),
        "oct_export": (i32, [vp, vp, vp]), "oct_upload": (i32, [vp, vp, vp]), "oct_counters": (i32, [vp, vp, vp]),
        "oct_mcs": (i32, [vp, C.POINTER(u64)]), "oct_destroy": (i32, [vp]),
        "oct_strerror": (C.c_char_p, [i32]), "oct_last_error": (C.c_char_p, [vp]),
        "oct_launch_count": (i32, [vp, C.POINTER(u64)]),
        "oct_w2_from_sums": (dbl, [u32, i64, i64]), "oct_c_from_sums": (dbl, [u32, i64, i64, i64]),
        "oct_time_per_sweep": (dbl, [u32, i32]), "oct_scheme_supported": (i32, [u32, i32]),
        "oct_set_option": (i32, [vp, i32, i32]),
        "oct_slope_autocorr": (i32, [vp, vp, vp, vp]), "oct_cs_from_sums": (dbl, [u64, i64, i64, i64]),
        "oct_observe": (i32, [vp, i32, vp, vp, vp, vp]), "oct_fetch": (i32, [vp, vp, vp, sz, vp]),
        "oct_observe_batch": (i32, [C.POINTER(vp), u32, i32, C.POINTER(vp), C.POINTER(vp), vp, vp]),
        "oct_width2_static": (i32, [vp, u32, i64, i64, vp, vp]),
    }
    for name in EXPORTS:
        fn = getattr(L, name)          # AttributeError if a declared symbol is not exported
        fn.restype, fn.argtypes = sig[name]
    _lib = L
    return L


def _strerror(code: int) -> str:
    try:
        return load().oct_strerror(code).decode()
    except Exception:
        return "?"


# ---- plain functions, one per C entry point ----------------------------------------------------------
def oct_lattice_bytes(L: int) -> int:
    return int(load().oct_lattice_bytes(L))


def oct_workspace_bytes(L: int) -> int:
    return int(load().oct_workspace_bytes(L))


def oct_scheme_supported(L: int, scheme: int) -> bool:
    return load().oct_scheme_supported(L, scheme) == OCT_OK


def oct_w2_from_sums(L: int, S1: int, S2: int) -> float:
    return float(load().oct_w2_from_sums(L, S1, S2))


def oct_c_from_sums(L: int, St: int, Ss: int, Sts: int) -> float:
    return float(load().oct_c_from_sums(L, St, Ss, Sts))


def oct_cs_from_sums(M: int, n11: int, n1t: int, n1s: int) -> float:
    return float(load().oct_cs_from_sums(M, n11, n1t, n1s))


def oct_time_per_sweep(L: int, scheme: int) -> float:
    return float(load().oct_time_per_sweep(L, scheme))


def _stream_ptr(stream) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def oct_sweep_batch(sims, n_mcs: int, p: float, q: float, scheme: int, stream=None):
    """n_mcs sweeps of every simulation in `sims` (one lattice size), all members in each kernel launch."""
    sims = list(sims)
    arr = (C.c_void_p * len(sims))(*[s._h for s in sims])
    rc = load().oct_sweep_batch(arr, len(sims), n_mcs, p, q, scheme, _stream_ptr(stream))
    if rc:
        raise OctError(rc, "oct_sweep_batch", load().oct_last_error(sims[0]._h).decode() if sims else "")


def oct_observe_batch(sims, what: int, snapshots=None, anchors=None, out=None, stream=None):
    """oct_observe for every simulation in `sims` (one lattice size) in three launches per 64 members; out: (n, 16) int64."""
    sims = list(sims)
    n = len(sims)
    if out is None:
        out = sims[0].torch.empty((n, 16), dtype=sims[0].torch.int64, device=sims[0].device)
    hs = (C.c_void_p * n)(*[s._h for s in sims])
    sp = (C.c_void_p * n)(*[t.data_ptr() for t in snapshots]) if snapshots is not None else None
    ap = (C.c_void_p * n)(*[t.data_ptr() for t in anchors]) if anchors is not None else None
    rc = load().oct_observe_batch(hs, n, what, sp, ap, out.data_ptr(), _stream_ptr(stream))
    if rc:
        raise OctError(rc, "oct_observe_batch", load().oct_last_error(sims[0]._h).decode() if sims else "")
    return out


def oct_width2_static(lattice, L: int, h00: int, net: int, out, stream=None):
    """oct_width2's sums {S1, S2, c, net} of the packed lattice in the CUDA tensor `lattice`, written to the int64[4] CUDA
    tensor `out` -- without a handle or workspace.  For callers that may not allocate device memory (see include/oct.h):
    the C call allocates nothing, and neither does this wrapper, which is why `out` has no default.  L <= 2^16
    (OctError with code OCT_ETOOBIG beyond); calls that can overlap on the GPU share one scratch array and race."""
    rc = load().oct_width2_static(lattice.data_ptr(), L, h00, net, out.data_ptr(), _stream_ptr(stream))
    if rc:
        raise OctError(rc, "oct_width2_static")
    return out


class Sim:
    """A simulation handle plus the torch-owned device buffers it runs on."""

    def __init__(self, L: int, seed: int, init: int = wl.INIT_FLAT, device="cuda:0", lattice=None):
        import torch
        self._l = load()
        if not torch.cuda.is_available():
            raise OctError(OCT_ECUDA, "Sim", "no CUDA device: liboct_b200 has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nb, nw = oct_lattice_bytes(L), oct_workspace_bytes(L)
        if nb == 0:
            raise OctError(OCT_EINVAL, "oct_lattice_bytes", f"L={L}")
        self.L = L
        self.seed = seed
        if lattice is not None:
            assert lattice.dtype == torch.int32 and lattice.numel() * 4 == nb and lattice.is_cuda
            self.lattice = lattice
            init = wl.INIT_FROM_DEVICE
        else:
            self.lattice = torch.empty(nb // 4, dtype=torch.int32, device=self.device)
        self.workspace = torch.empty(nw, dtype=torch.uint8, device=self.device)
        self._h = C.c_void_p()
        rc = self._l.oct_create(C.byref(self._h), L, seed, init, self.lattice.data_ptr(), self.workspace.data_ptr(),
                                _stream_ptr(None))
        if rc:
            raise OctError(rc, "oct_create")

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            self._l.oct_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, where: str):
        if rc:
            raise OctError(rc, where, self._l.oct_last_error(self._h).decode())

    # -- C entry points
    def oct_sweep(self, n_mcs: int, p: float, q: float, scheme: int, stream=None):
        self._check(self._l.oct_sweep(self._h, n_mcs, p, q, scheme, _stream_ptr(stream)), "oct_sweep")

    def oct_set_state(self, t: int, h00: int, net: int, stream=None):
        self._check(self._l.oct_set_state(self._h, t, h00, net, _stream_ptr(stream)), "oct_set_state")

    def oct_heights(self, out=None, stream=None):
        if out is None:
            out = self.torch.empty((self.L, self.L), dtype=self.torch.int32, device=self.device)
        self._check(self._l.oct_heights(self._h, out.data_ptr(), _stream_ptr(stream)), "oct_heights")
        return out

    def oct_width2(self, out=None, stream=None):
        """Device tensor int64[4] = {S1, S2, c, net}."""
        if out is None:
            out = self.torch.empty(4, dtype=self.torch.int64, device=self.device)
        self._check(self._l.oct_width2(self._h, out.data_ptr(), _stream_ptr(stream)), "oct_width2")
        return out

    def oct_snapshot(self, lattice_copy=None, anchor=None, stream=None):
        if lattice_copy is None:
            lattice_copy = self.torch.empty_like(self.lattice)
        if anchor is None:
            anchor = self.torch.empty(2, dtype=self.torch.int64, device=self.device)
        self._check(self._l.oct_snapshot(self._h, lattice_copy.data_ptr(), anchor.data_ptr(), _stream_ptr(stream)),
                    "oct_snapshot")
        return lattice_copy, anchor

    def oct_autocorr(self, snapshot, anchor, out=None, stream=None):
        """Device tensor int64[5] = {S_t, S_s, S_ts, c_t, c_s}."""
        if out is None:
            out = self.torch.empty(5, dtype=self.torch.int64, device=self.device)
        self._check(self._l.oct_autocorr(self._h, snapshot.data_ptr(), anchor.data_ptr(), out.data_ptr(),
                                         _stream_ptr(stream)), "oct_autocorr")
        return out

    def oct_slope_autocorr(self, snapshot, out=None, stream=None):
        """Device tensor int64[6] = {sum nx_t nx_s, sum ny_t ny_s, sum nx_t, sum ny_t, sum nx_s, sum ny_s}."""
        if out is None:
            out = self.torch.empty(6, dtype=self.torch.int64, device=self.device)
        self._check(self._l.oct_slope_autocorr(self._h, snapshot.data_ptr(), out.data_ptr(), _stream_ptr(stream)),
                    "oct_slope_autocorr")
        return out

    def oct_observe(self, what: int, snapshot=None, anchor=None, out=None, stream=None):
        """Device tensor int64[16]: [0..3] W^2 sums, [4..8] C_h sums, [9..14] C_s sums (one pass, see oct.h)."""
        if out is None:
            out = self.torch.empty(16, dtype=self.torch.int64, device=self.device)
        self._check(self._l.oct_observe(self._h, what, snapshot.data_ptr() if snapshot is not None else None,
                                        anchor.data_ptr() if anchor is not None else None, out.data_ptr(), _stream_ptr(stream)),
                    "oct_observe")
        return out

    def oct_fetch(self, src, host_ptr: int, nbytes: int, stream=None):
        self._check(self._l.oct_fetch(self._h, src.data_ptr(), host_ptr, nbytes, _stream_ptr(stream)), "oct_fetch")

    def oct_export(self, host=None, stream=None) -> np.ndarray:
        """Canonical packed words as a (L/4, L/4) uint32 numpy array (synchronises)."""
        n = self.L // 4
        if host is None:
            host = np.empty((n, n), dtype=np.uint32)
        self._check(self._l.oct_export(self._h, host.ctypes.data, _stream_ptr(stream)), "oct_export")
        return host

    def oct_export_to(self, host_ptr: int, stream=None):
        self._check(self._l.oct_export(self._h, host_ptr, _stream_ptr(stream)), "oct_export")

    def oct_upload(self, host, stream=None):
        ptr = host.ctypes.data if isinstance(host, np.ndarray) else int(host)
        if isinstance(host, np.ndarray):
            assert host.dtype == np.uint32 and host.size * 4 == oct_lattice_bytes(self.L) and host.flags.c_contiguous
        self._check(self._l.oct_upload(self._h, ptr, _stream_ptr(stream)), "oct_upload")

    def oct_counters(self, stream=None):
        """(h00, net) read back from the device (synchronises)."""
        o = np.zeros(2, dtype=np.int64)
        self._check(self._l.oct_counters(self._h, o.ctypes.data, _stream_ptr(stream)), "oct_counters")
        return int(o[0]), int(o[1])

    def oct_set_option(self, option: int, value: int):
        self._check(self._l.oct_set_option(self._h, option, value), "oct_set_option")

    def oct_mcs(self) -> int:
        t = C.c_uint64()
        self._check(self._l.oct_mcs(self._h, C.byref(t)), "oct_mcs")
        return int(t.value)

    def oct_launch_count(self) -> int:
        n = C.c_uint64()
        self._check(self._l.oct_launch_count(self._h, C.byref(n)), "oct_launch_count")
        return int(n.value)
