"""CPU oracle for the octahedron-model DD sweep of arXiv 1705.01022 -- TEST INFRASTRUCTURE ONLY.

Thin ctypes wrapper around ``oracle/oct_oracle.c`` (plain single-threaded C, written from PAPER.md and
the readings in DESIGN.md).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product
(``paper_1705_01022_b200``) never does, and this package never imports the product.

The exact rational observables (W^2, C_h) are formed here with Python integers / Fractions from the
integer sums (Eq. (3), Eq. (6) PAPER.md:92-98 with readings R6/R7 of DESIGN.md).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from fractions import Fraction

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oct_oracle.c")
_LIB = os.path.join(_HERE, "liboct_oracle.so")

# scheme encoding of include/oct.h (restated, not shared): dev | blk<<4 | tcx<<8 | tcy<<12 | log2D<<16 | ka<<21 | w<<23
DEV_DTR, DEV_DT, DEV_DB, DEV_CDB, DEV_DBH = 0, 1, 2, 3, 4
BLK_DB, BLK_DB_DELAYED, BLK_DT, BLK_DTR = 0, 1, 2, 3


def scheme(dev: int, blk: int, log2D: int, tcx: int = 1, tcy: int = 1, ka: int = 0, w: int = 0) -> int:
    """ka: t_async = 2^-ka MCS; w: explicit dead-border width (0 = the scheme's own) -- dead-border device layers only."""
    return dev | (blk << 4) | (tcx << 8) | (tcy << 12) | (log2D << 16) | (ka << 21) | (w << 23)


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, no OpenMP, no -march flags)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class TraceRec(C.Structure):
    _fields_ = [("x", C.c_uint32), ("y", C.c_uint32), ("t", C.c_uint32), ("set", C.c_uint32),
                ("dom", C.c_uint32), ("k", C.c_uint32), ("cell", C.c_uint32), ("cls", C.c_int32),
                ("result", C.c_int32)]


TRACE_DTYPE = np.dtype([("x", "<u4"), ("y", "<u4"), ("t", "<u4"), ("set", "<u4"), ("dom", "<u4"),
                        ("k", "<u4"), ("cell", "<u4"), ("cls", "<i4"), ("result", "<i4")])

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, u32, u64, i64, dbl, i32 = C.c_void_p, C.c_uint32, C.c_uint64, C.c_int64, C.c_double, C.c_int
        L.orc_philox4x32_10.argtypes = [vp, vp, vp]; L.orc_philox4x32_10.restype = None
        L.orc_create.argtypes = [u32, u64, i32, i32]; L.orc_create.restype = vp
        L.orc_destroy.argtypes = [vp]; L.orc_destroy.restype = None
        L.orc_clone.argtypes = [vp]; L.orc_clone.restype = vp
        L.orc_lattice.argtypes = [vp]; L.orc_lattice.restype = vp
        L.orc_tracked_heights.argtypes = [vp]; L.orc_tracked_heights.restype = vp
        L.orc_mcs.argtypes = [vp]; L.orc_mcs.restype = u64
        L.orc_net.argtypes = [vp]; L.orc_net.restype = i64
        L.orc_h00.argtypes = [vp]; L.orc_h00.restype = i64
        L.orc_set_time.argtypes = [vp, u64]; L.orc_set_time.restype = None
        L.orc_set_anchor.argtypes = [vp, i64, i64]; L.orc_set_anchor.restype = None
        L.orc_set_shuffle.argtypes = [vp, u64]; L.orc_set_shuffle.restype = None
        L.orc_set_filter.argtypes = [vp, i32, u32, u32, u32, u32]; L.orc_set_filter.restype = None
        L.orc_set_trace.argtypes = [vp, vp, u64]; L.orc_set_trace.restype = None
        L.orc_trace_count.argtypes = [vp]; L.orc_trace_count.restype = u64
        L.orc_prob16.argtypes = [dbl]; L.orc_prob16.restype = u32
        L.orc_attempt.argtypes = [vp, u32, u32, u32, u32, u32]; L.orc_attempt.restype = i32
        L.orc_sweep_rs.argtypes = [vp, u64, dbl, dbl]; L.orc_sweep_rs.restype = i32
        L.orc_sweep_dd.argtypes = [vp, u64, dbl, dbl, u32]; L.orc_sweep_dd.restype = i32
        L.orc_check_scheme.argtypes = [u32, u32]; L.orc_check_scheme.restype = i32
        L.orc_mcs_control.argtypes = [u64, u32, u32, u32, vp]; L.orc_mcs_control.restype = None
        L.orc_heights.argtypes = [vp, vp]; L.orc_heights.restype = None
        L.orc_heights_rowpath.argtypes = [vp, vp]; L.orc_heights_rowpath.restype = None
        L.orc_sums.argtypes = [vp, vp]; L.orc_sums.restype = i32
        L.orc_sums_rowpath.argtypes = [vp, vp]; L.orc_sums_rowpath.restype = i32
        L.orc_autocorr_sums.argtypes = [vp, vp, vp]; L.orc_autocorr_sums.restype = i32
        L.orc_slope_autocorr_sums.argtypes = [vp, vp, vp]; L.orc_slope_autocorr_sums.restype = i32
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return o


def prob16(p: float) -> int:
    return int(lib().orc_prob16(float(p)))


def mcs_control(seed: int, t: int, L: int, dev: int):
    """(Ox, Oy, perm) of MCS t."""
    o = np.zeros(6, dtype=np.uint32)
    lib().orc_mcs_control(seed, t, L, dev, o.ctypes.data)
    return int(o[0]), int(o[1]), tuple(int(v) for v in o[2:6])


def w2_from_sums(L: int, S1: int, S2: int) -> Fraction:
    """W^2 = <h^2> - <h>^2 over the L^2 sites (Eq. (3), reading R6), exact."""
    N = L * L
    return Fraction(N * int(S2) - int(S1) ** 2, N * N)


def c_from_sums(L: int, St: int, Ss: int, Sts: int) -> Fraction:
    """C_h(t,s) = <h_t h_s> - <h_t><h_s> (Eq. (6), reading R7), exact."""
    N = L * L
    return Fraction(N * int(Sts) - int(St) * int(Ss), N * N)


class Oracle:
    """One simulated lattice."""

    def __init__(self, L: int, seed: int, init: int = 0, track_heights: bool = False, _handle=None):
        self._l = lib()
        self.L = L
        self.seed = seed
        self._h = _handle if _handle is not None else self._l.orc_create(L, seed, init, int(track_heights))
        if not self._h:
            raise ValueError(f"orc_create failed for L={L}, init={init}")
        self._trace_buf = None

    def close(self):
        if self._h:
            self._l.orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state -------------------------------------------------------------------------------
    @property
    def lattice(self) -> np.ndarray:
        """View of the canonical packed words, shape (L/4, L/4), uint32."""
        n = self.L // 4
        buf = (C.c_uint32 * (n * n)).from_address(self._l.orc_lattice(self._h))
        return np.frombuffer(buf, dtype=np.uint32).reshape(n, n)

    def set_lattice(self, words: np.ndarray, h00: int = 0, net: int = 0, t: int | None = None):
        self.lattice[...] = np.asarray(words, dtype=np.uint32).reshape(self.L // 4, self.L // 4)
        self._l.orc_set_anchor(self._h, h00, net)
        if t is not None:
            self._l.orc_set_time(self._h, t)

    @property
    def tracked_heights(self) -> np.ndarray:
        p = self._l.orc_tracked_heights(self._h)
        if not p:
            raise ValueError("created without track_heights")
        buf = (C.c_int32 * (self.L * self.L)).from_address(p)
        return np.frombuffer(buf, dtype=np.int32).reshape(self.L, self.L)

    @property
    def t(self) -> int:
        return int(self._l.orc_mcs(self._h))

    @property
    def net(self) -> int:
        return int(self._l.orc_net(self._h))

    @property
    def h00(self) -> int:
        return int(self._l.orc_h00(self._h))

    def clone(self) -> "Oracle":
        h = self._l.orc_clone(self._h)
        if not h:
            raise MemoryError
        return Oracle(self.L, self.seed, _handle=h)

    # ---- test hooks --------------------------------------------------------------------------
    def set_shuffle(self, seed: int):
        self._l.orc_set_shuffle(self._h, seed)

    def set_filter(self, on: bool, x0=0, y0=0, w=0, h=0):
        self._l.orc_set_filter(self._h, int(on), x0, y0, w, h)

    def start_trace(self, capacity: int):
        self._trace_buf = np.zeros(capacity, dtype=TRACE_DTYPE)
        self._l.orc_set_trace(self._h, self._trace_buf.ctypes.data, capacity)

    def stop_trace(self) -> np.ndarray:
        n = int(self._l.orc_trace_count(self._h))
        buf = self._trace_buf
        self._l.orc_set_trace(self._h, None, 0)
        self._trace_buf = None
        if n > len(buf):
            raise OverflowError(f"trace overflow: {n} > {len(buf)}")
        return buf[:n]

    # ---- dynamics ----------------------------------------------------------------------------
    def attempt(self, x: int, y: int, r16: int, P16: int, Q16: int) -> int:
        return int(self._l.orc_attempt(self._h, x, y, r16, P16, Q16))

    def sweep_rs(self, n_mcs: int, p: float, q: float):
        rc = self._l.orc_sweep_rs(self._h, n_mcs, p, q)
        if rc:
            raise RuntimeError(f"orc_sweep_rs -> {rc}")

    def sweep(self, n_mcs: int, p: float, q: float, scheme_code: int):
        rc = self._l.orc_sweep_dd(self._h, n_mcs, p, q, scheme_code)
        if rc:
            raise ValueError(f"orc_sweep_dd -> {rc}")

    # ---- observables -------------------------------------------------------------------------
    def heights(self, rowpath: bool = False) -> np.ndarray:
        out = np.empty((self.L, self.L), dtype=np.int32)
        (self._l.orc_heights_rowpath if rowpath else self._l.orc_heights)(self._h, out.ctypes.data)
        return out

    def sums(self, rowpath: bool = False):
        """(S1, S2, c, net) with c = h(0,0).  rowpath: integrate up column 0 and along the rows, streaming (no
        height array; the only form that fits in memory at L = 2^17)."""
        o = np.zeros(4, dtype=np.int64)
        rc = (self._l.orc_sums_rowpath if rowpath else self._l.orc_sums)(self._h, o.ctypes.data)
        if rc:
            raise MemoryError
        return tuple(int(v) for v in o)

    def w2(self) -> Fraction:
        S1, S2, _, _ = self.sums()
        return w2_from_sums(self.L, S1, S2)

    def mean_height(self) -> Fraction:
        S1, _, c, _ = self.sums()
        return Fraction(c) + Fraction(S1, self.L * self.L)

    def autocorr_sums(self, snap: "Oracle"):
        """(S_t, S_s, S_ts, c_t, c_s) against a snapshot taken at waiting time s."""
        o = np.zeros(5, dtype=np.int64)
        rc = self._l.orc_autocorr_sums(self._h, snap._h, o.ctypes.data)
        if rc:
            raise RuntimeError(f"orc_autocorr_sums -> {rc}")
        return tuple(int(v) for v in o)

    def slope_autocorr_sums(self, snap: "Oracle"):
        """(sum nx_t nx_s, sum ny_t ny_s, sum nx_t, sum ny_t, sum nx_s, sum ny_s) against a snapshot."""
        o = np.zeros(6, dtype=np.int64)
        rc = self._l.orc_slope_autocorr_sums(self._h, snap._h, o.ctypes.data)
        if rc:
            raise RuntimeError(f"orc_slope_autocorr_sums -> {rc}")
        return tuple(int(v) for v in o)

    def c_s(self, snap: "Oracle") -> Fraction:
        """C_s(t,s) over all 2 L^2 slope variables, exact."""
        xx, yy, xt, yt, xs, ys = self.slope_autocorr_sums(snap)
        M = 2 * self.L * self.L
        return Fraction(M * (xx + yy) - (xt + yt) * (xs + ys), M * M)

    def c_h(self, snap: "Oracle") -> Fraction:
        St, Ss, Sts, _, _ = self.autocorr_sums(snap)
        return c_from_sums(self.L, St, Ss, Sts)
