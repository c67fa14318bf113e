#!/usr/bin/env python
"""Small invocation of every kernel of libgg (both dtypes, ragged multi-tile grids, a batch, ghost
rows and domain edges) meant to be run under compute-sanitizer on the GPU box:

    compute-sanitizer --tool memcheck  python tests/sanitizer_run.py
    compute-sanitizer --tool racecheck python tests/sanitizer_run.py
    compute-sanitizer --tool synccheck python tests/sanitizer_run.py
    compute-sanitizer --tool initcheck python tests/sanitizer_run.py

It also checks every result against the CPU oracle, so a clean sanitizer log is a log of correct
runs.  Not a pytest file (the sanitizers slow the kernels down 10-100x).  Round 1: compute-sanitizer
is closed on the GPU pool this was developed on ("runs under it have left GPUs needing a reset"),
so only the plain run (all twelve kernel x dtype cases correct) has been made; the kernels' own
guards are the bounded mbarrier / flag spins that trap instead of hanging."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2006_01748_b200 import binding, workloads  # noqa: E402

KERNELS = {"generic": binding.GG_KERNEL_GENERIC, "stream": binding.GG_KERNEL_STREAM,
           "stream2": binding.GG_KERNEL_STREAM2, "pair": binding.GG_KERNEL_PAIR,
           "quad": binding.GG_KERNEL_QUAD, "resident": binding.GG_KERNEL_RESIDENT}


def main():
    worst = 0.0
    for dtype, tol in (("f64", 1e-10), ("f32", 2e-4)):
        wl = workloads.random_problem(11, 488 if dtype == "f64" else 976, 45, batch=2)
        n = 7
        ref = [oracle.step(wl.U[s], wl.V[s], wl.W[s], wl.a, wl.b, wl.c, r=wl.r[s], d=wl.d[s],
                           alpha=wl.alpha[s], c_r=wl.c_r[s], n=n, dt=wl.dt, dx=wl.h) for s in range(2)]
        for name, k in KERNELS.items():
            with binding.from_workload(wl, dtype=dtype) as sim:
                sim.set_option(binding.GG_OPT_KERNEL, k)
                sim.step(n, wl.dt)
                diag = sim.diagnostics(1e-2)
                dt, lam = sim.max_stable_dt(0.2)
                got = sim.get_state_numpy()
            err = max(float(np.max(np.abs(got[f][s].astype(np.float64) - ref[s][f])))
                      for f in range(3) for s in range(2))
            print(f"{dtype} {name}: max-abs err {err:.2e}", flush=True)
            assert err <= tol and np.isfinite(diag).all() and dt > 0 and lam > 0
            worst = max(worst, err)
    print("sanitizer_run OK")


if __name__ == "__main__":
    main()
