"""Builds paper_1812_02647_b200/libhs.so (the C-ABI library of include/hs.h) in-tree with nvcc for sm_100a.

    python -m paper_1812_02647_b200.build [--force] [-v] [--tuning]

One object per .cu (compiled in parallel), then one shared library.  nvcc cross-compiles without a GPU.
--tuning builds libhs_tuning.so instead: the same sources with -DHS_TUNING, the only build in which the kernels'
schedule parameters (ring sizes, lags, spin limit) can be overridden through HS_* environment variables.  The product
library reads no environment variable; the tuning build serves the builder's sweeps and the forced-timeout test.
"""
from __future__ import annotations

import concurrent.futures
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libhs.so")
LIB_TUNING = os.path.join(HERE, "libhs_tuning.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC,-Wall,-Wextra", "--expt-relaxed-constexpr"]


def _deps():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(HERE, "..", "include", "*.h"))


def _stale(target, sources):
    return (not os.path.exists(target)) or any(os.path.getmtime(s) > os.path.getmtime(target) for s in sources)


def _compile(src, verbose, tuning=False):
    obj = os.path.join(OBJ, os.path.basename(src)[:-3] + (".tuning.o" if tuning else ".o"))
    if _stale(obj, [src] + _deps()):
        extra = (["-DHS_TUNING"] + os.environ.get("HS_TUNING_NVCC_FLAGS", "").split()) if tuning else []
        cmd = [NVCC] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            sys.stderr.write(r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False, tuning: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    lib = LIB_TUNING if tuning else LIB
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    if force:
        for f in glob.glob(os.path.join(OBJ, "*.tuning.o" if tuning else "*.o")):
            if tuning or not f.endswith(".tuning.o"):
                os.remove(f)
    with concurrent.futures.ThreadPoolExecutor(max_workers=min(os.cpu_count() or 4, len(srcs))) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose, tuning), srcs))
    if force or _stale(lib, objs):
        tmp = lib + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC, "-shared", "-o", tmp] + objs)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, tuning="--tuning" in sys.argv))
