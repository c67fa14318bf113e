"""Build step for libgg.so, the product's C-ABI CUDA library (include/gg.h).

    nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -Xcompiler -fPIC -Xfatbin -compress-all
         -c --threads 6
         csrc/gg_api.cu csrc/gg3_api.cu csrc/gg_noalloc.cu csrc/gg_inst_{quad,pair,stream,stream2}.cu
    nvcc -shared -cudart static *.o -o paper_2006_01748_b200/libgg.so

(gg3_api.cu: the three-dimensional extension, include/gg3.h; gg_noalloc.cu: the allocation-free
diagnostics call with its built-in device scratch; gg_inst_*.cu: the builds of the step
kernels, one translation unit per family so that they compile in parallel.)

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
# translation units: the two ABIs and one per family of step-kernel builds (compiled in parallel)
TUS = [os.path.join(CSRC, f) for f in ("gg_api.cu", "gg3_api.cu", "gg_noalloc.cu", "gg_inst_quad.cu",
                                       "gg_inst_pair.cu", "gg_inst_stream.cu", "gg_inst_stream2.cu")]


def sources():
    return (sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.inc")))
            + [os.path.join(ROOT, "include", "gg.h"), os.path.join(ROOT, "include", "gg3.h")])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def commands(out: str, objdir: str, extra=()):
    """Compile every translation unit to an object (in parallel), then link the shared library."""
    flags = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++20",
             "-Xcompiler", "-fPIC", "-Xfatbin", "-compress-all", *extra]
    objs = [os.path.join(objdir, os.path.splitext(os.path.basename(t))[0] + ".o") for t in TUS]
    return ([*flags, "-c", "--threads", str(len(TUS)), "-odir", objdir, *TUS],
            [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static", *objs, "-o", out])


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        import shutil
        import tempfile
        tmp = LIB + f".tmp{os.getpid()}"
        objdir = tempfile.mkdtemp(prefix="gg_build_")
        try:
            for cmd in commands(tmp, objdir, ("-Xptxas", "-v") if verbose else ()):
                subprocess.run(cmd, check=True)
            os.replace(tmp, LIB)
        finally:
            shutil.rmtree(objdir, ignore_errors=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
