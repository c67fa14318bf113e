"""Build step for the CPU oracle (TEST INFRASTRUCTURE, not product code).

Compiles oracle/gg_oracle.cpp and oracle/gg3_oracle.cpp (the 3-D extension) into
oracle/libgg_oracle.so with
    g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC
(-ffp-contract=off: no FMA contraction, so the arithmetic is exactly what the source spells out).
Called by `oracle.load()` when the library is missing or older than its source, and by
`__graft_entry__.build()` ("building the checker is not using it").
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "gg_oracle.cpp"), os.path.join(HERE, "gg3_oracle.cpp")]
LIB = os.path.join(HERE, "libgg_oracle.so")


def needs_build() -> bool:
    return (not os.path.exists(LIB)) or any(os.path.getmtime(LIB) < os.path.getmtime(s) for s in SRCS)


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c++17", "-shared", "-fPIC",
               "-Wall", "-Wextra", *SRCS, "-o", tmp]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)  # atomic: concurrent test workers never see a half-written file
    return LIB


if __name__ == "__main__":
    print(build(force=True))
