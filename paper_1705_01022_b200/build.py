"""Build liboct_b200.so (the C-ABI product library) in-tree with nvcc for sm_100a.

    python -m paper_1705_01022_b200.build [ptxas_report.txt]
"""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liboct_b200.so")
SOURCES = ["oct_api.cu"]
HEADERS = ["sweep.cuh", "sweep_links.cuh", "observe.cuh", "observe_rows.cuh", "philox.cuh", os.path.join("..", "..", "include", "oct.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-Wall", "-shared", "--use_fast_math", "-Xptxas", "-v"]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built")
    return exe


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, ptxas_info: str | None = None) -> str:
    """ptxas_info: optional path that receives ptxas' per-kernel register / spill / shared-memory report."""
    if force or stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc(), *NVCC_FLAGS, "-o", tmp, *[os.path.join(CSRC, s) for s in SOURCES]]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode:
            print(res.stdout)
            print(res.stderr)
        if res.returncode:
            raise RuntimeError("nvcc failed:\n" + res.stderr[-4000:])
        if ptxas_info:
            with open(ptxas_info, "w") as f:
                f.write("".join(l for l in res.stderr.splitlines(True) if "Compile time" not in l))
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=False, ptxas_info=sys.argv[1] if len(sys.argv) > 1 else None))
