"""python -m paper_1812_02647_b200.microbench — builds hs_microbench.cu for sm_100a and runs it on cuda:0.

Prints the hardware rates DESIGN.md section 6 uses as secondary roofs (distributed-shared-memory gather bandwidth per
cluster size, scattered-sector load rates, dirty-L2 residency of a rewritten ring).  Not part of libhs.so.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build() -> str:
    exe = os.path.join(HERE, "hs_microbench")
    src = os.path.join(HERE, "hs_microbench.cu")
    if not os.path.exists(exe) or os.path.getmtime(exe) < os.path.getmtime(src):
        subprocess.check_call([NVCC, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                               "-o", exe, src])
    return exe


if __name__ == "__main__":
    exe = build()
    if "--build-only" not in sys.argv:
        sys.exit(subprocess.call([exe]))
