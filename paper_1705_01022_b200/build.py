"""Build liboct_b200.so (the C-ABI product library) in-tree with nvcc for sm_100a.

    python -m paper_1705_01022_b200.build [ptxas_report.txt]
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liboct_b200.so")
# translation units: (object name, source, extra defines).  sweep_inst.cu is compiled once per kernel family and
# domain size so that the ~200 kernel instantiations build in parallel.
UNITS = [("oct_api", "oct_api.cu", []), ("width2_static", "width2_static.cu", [])] + \
        [(f"packed_{ld}", "sweep_inst.cu", ["-DOCT_INST_FAMILY=0", f"-DOCT_INST_LOG2D={ld}"]) for ld in (5, 6, 7, 8)] + \
        [(f"links_{ld}", "sweep_inst.cu", ["-DOCT_INST_FAMILY=1", f"-DOCT_INST_LOG2D={ld}"]) for ld in (5, 6, 7, 8)]
HEADERS = ["sweep.cuh", "sweep_links.cuh", "observe.cuh", "observe_rows.cuh", "philox.cuh", "launch.h", "sweep_inst.cu", "oct_api.cu", "width2_static.cu",
           os.path.join("..", "..", "include", "oct.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2,-Wall", "--use_fast_math", "-Xptxas", "-v"]
OBJDIR = os.path.join(HERE, "build")


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built")
    return exe


STAMP = LIB + ".flags"      # hash of the flags the library on disk was built with (absent: the default flags)


def _flags_hash(extra_flags=()) -> str:
    return hashlib.sha256(" ".join([*NVCC_FLAGS, *extra_flags]).encode()).hexdigest()[:12]


def stale() -> bool:
    """True if the library is missing, older than a source, or was linked from an experiment build (extra_flags)."""
    if not os.path.exists(LIB):
        return True
    if os.path.exists(STAMP) and open(STAMP).read().strip() != _flags_hash():
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


# what each translation unit includes: a unit is recompiled when one of these (or this file) is newer than its object
UNIT_DEPS = {"oct_api.cu": ["oct_api.cu", "observe.cuh", "observe_rows.cuh", "philox.cuh", "launch.h", "sweep.cuh",
                            os.path.join("..", "..", "include", "oct.h")],
             "width2_static.cu": ["width2_static.cu", "observe.cuh", "observe_rows.cuh", os.path.join("..", "..", "include", "oct.h")],
             "sweep_inst.cu": ["sweep_inst.cu", "launch.h", "sweep.cuh", "sweep_links.cuh", "philox.cuh"]}


def _unit_stale(obj: str, src: str, force: bool) -> bool:
    if force or not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    deps = [os.path.join(CSRC, f) for f in UNIT_DEPS[src]] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, ptxas_info: str | None = None, extra_flags=()) -> str:
    """Compile the stale units (in parallel; all of them with force=True), link liboct_b200.so.  Objects are kept under
    build/<flags hash>/ (git-ignored) so that a change to one header recompiles only the units that include it, and a build
    with extra_flags (always linked, even when the default library is up to date) never shares objects with the default one.
    ptxas_info: optional path that receives ptxas' per-kernel register / spill / shared-memory report of the units that
    were compiled; extra_flags: additional nvcc flags (e.g. -D switches)."""
    if not (force or extra_flags or stale()):
        return LIB
    # objects live under build/<hash of every flag that shapes them>: an experiment build (extra_flags) can never leave
    # objects behind that a later default build would take for its own
    objdir = os.path.join(OBJDIR, _flags_hash(extra_flags))
    os.makedirs(objdir, exist_ok=True)
    tag = f".tmp{os.getpid()}"
    procs, objs = [], []
    for name, src, defs in UNITS:
        obj = os.path.join(objdir, name + ".o")
        objs.append(obj)
        if _unit_stale(obj, src, force):
            cmd = [nvcc(), *NVCC_FLAGS, *defs, *extra_flags, "-c", "-o", obj + tag, os.path.join(CSRC, src)]
            procs.append((name, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    report, failed = [], None
    for name, obj, pr in procs:
        out, err = pr.communicate()
        report.append(err)
        if verbose or pr.returncode:
            print(out)
            print(err)
        if pr.returncode:
            if failed is None:
                failed = f"nvcc failed on {name}:\n" + err[-4000:]
            if os.path.exists(obj + tag):
                os.unlink(obj + tag)
        else:
            os.replace(obj + tag, obj)
    if failed:
        raise RuntimeError(failed)
    tmp = LIB + tag
    res = subprocess.run([nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", tmp, *objs], capture_output=True, text=True)
    if res.returncode:
        raise RuntimeError("link failed:\n" + res.stderr[-4000:])
    if ptxas_info:
        with open(ptxas_info, "w") as f:
            f.write("".join(l for e in report for l in e.splitlines(True) if "Compile time" not in l))
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(_flags_hash(extra_flags) + "\n")
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose=False, ptxas_info=sys.argv[1] if len(sys.argv) > 1 else None))
