"""Build step for libgg.so, the product's C-ABI CUDA library (include/gg.h).

    nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
         paper_2006_01748_b200/csrc/gg_api.cu paper_2006_01748_b200/csrc/gg3_api.cu
         -o paper_2006_01748_b200/libgg.so

(gg3_api.cu: the three-dimensional extension, include/gg3.h.)

nvcc cross-compiles without a GPU; the CUDA runtime is linked statically and the one driver-API
symbol the library needs (cuTensorMapEncodeTiled) is resolved at run time through
cudaGetDriverEntryPoint, so the .so loads on a machine without libcuda (the CPU test tier checks
its exported symbols there).  The .so is built in-tree and is git-ignored.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgg.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def sources():
    return (sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")))
            + [os.path.join(ROOT, "include", "gg.h"), os.path.join(ROOT, "include", "gg3.h")])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def command(out: str, extra=()):
    return [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++20",
            "-shared", "-Xcompiler", "-fPIC", "-cudart", "static", *extra,
            os.path.join(CSRC, "gg_api.cu"), os.path.join(CSRC, "gg3_api.cu"), "-o", out]


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = command(tmp, ("-Xptxas", "-v") if verbose else ())
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
