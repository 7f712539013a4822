"""Build and run the sm_100a microbenchmarks behind DESIGN.md section 9 (TMEM read-out rate, UMMA shapes, TMA issue
costs, cluster occupancy).  Needs a B200:

    python -m paper_2606_05484_b200.microbench.run [name ...]

Each benchmark is a stand-alone .cu file in this directory that shares only csrc/tc_common.{cu,cuh} (the inline-PTX
wrappers) with the library; binaries go to a temporary directory.  Measurement tools: nothing in the library, the tests
or bench.py depends on them.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))
PKG = os.path.dirname(HERE)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def main(names):
    srcs = sorted(glob.glob(os.path.join(HERE, "*.cu")))
    if names:
        srcs = [s for s in srcs if os.path.basename(s)[:-3] in names]
    tmp = tempfile.mkdtemp(prefix="mapl_microbench_")
    for src in srcs:
        exe = os.path.join(tmp, os.path.basename(src)[:-3])
        cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-I", os.path.join(PKG, "csrc"),
               "-I", os.path.join(os.path.dirname(PKG), "include"), "-o", exe, src, os.path.join(PKG, "csrc", "tc_common.cu")]
        subprocess.run(cmd, check=True)
        print(f"== {os.path.basename(src)}", flush=True)
        subprocess.run([exe], check=False)


if __name__ == "__main__":
    main(sys.argv[1:])
