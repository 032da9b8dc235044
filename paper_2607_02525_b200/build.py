"""Build libpeek.so (hand-written CUDA for sm_100a) in-tree with nvcc; cross-compiles without a GPU.

    python -m paper_2607_02525_b200.build [--force] [-v] [--checked]
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpeek.so")
LIB_CHECKED = os.path.join(_HERE, "libpeek_checked.so")
SOURCES = ["peek_api.cu", "peek_hash.cu", "peek_lpm.cu", "peek_tree.cu", "peek_demand.cu", "peek_signals.cu", "peek_offline.cu",
           "peek_interleave.cu"]
HEADERS = ["peek_common.cuh", "peek_grid.cuh", "peek_sort.cuh", os.path.join("..", "..", "include", "peek.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-diag-suppress", "177"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    return "nvcc"


def _stale(out: str, deps) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(d) > t for d in deps)


def build_libpeek(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked=True builds libpeek_checked.so (-DPEEK_CHECKED: range checks on every index computed
    from device data, canaries around the workspace pieces); load it with PEEK_LIB=<path>."""
    hdrs = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    objdir = os.path.join(_HERE, "build_checked" if checked else "build")
    lib = LIB_CHECKED if checked else LIB
    extra = ["-DPEEK_CHECKED"] if checked else []
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(objdir, s.replace(".cu", ".o"))
        if force or _stale(obj, [src] + hdrs):
            jobs.append([nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj])

    def run(cmd):
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
        if verbose:
            sys.stderr.write(r.stderr)

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            list(ex.map(run, jobs))
    objs = [os.path.join(objdir, s.replace(".cu", ".o")) for s in SOURCES]
    if force or jobs or _stale(lib, objs):
        run([nvcc, "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"])
    return lib


if __name__ == "__main__":
    print(build_libpeek(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
