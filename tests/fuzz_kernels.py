#!/usr/bin/env python
"""Random-shape fuzz of every kernel of libgg against the CPU oracle AND against each other.

    python tests/fuzz_kernels.py [seed] [seconds] [--large]

Each case draws a dtype, a grid (widths around the kernels' tile widths -- 60, 118, 236, 240, 472,
480, 944 cells --, tiny and ragged heights), a batch, a step count, a mesh ratio dy/dx and sometimes
a chunking option; runs generic, stream, stream2, resident, pair and quad through the C ABI; asserts
the oracle tolerance (fp64 1e-10, fp32 2e-4) and that all kernels agree BIT FOR BIT.  Not a pytest
file (open-ended run time).  Round 1: 255 000 cases over seeds 1-3, 11, 12 (33 minutes), 0 failures.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2006_01748_b200 import binding as B, workloads  # noqa: E402

KERNELS = {"generic": B.GG_KERNEL_GENERIC, "stream": B.GG_KERNEL_STREAM, "stream2": B.GG_KERNEL_STREAM2,
           "resident": B.GG_KERNEL_RESIDENT, "pair": B.GG_KERNEL_PAIR, "quad": B.GG_KERNEL_QUAD}


def main():
    args = [a for a in sys.argv[1:] if not a.startswith("--")]
    large = "--large" in sys.argv
    rng = np.random.default_rng(int(args[0]) if args else 0)
    budget = float(args[1]) if len(args) > 1 else 120.0
    t0, ncase, bad = time.time(), 0, 0
    while time.time() - t0 < budget:
        dtype = str(rng.choice(["f64", "f32"]))
        c = 2 if dtype == "f64" else 4
        wide = rng.integers(300, 1500) if large else rng.integers(1, 700)
        tall = rng.integers(100, 700) if large else rng.integers(2, 400)
        nx = int(rng.choice([c, 2 * c, 60, 59 * c, 236, 240, 472, 480, 944, wide * c]))
        ny = int(rng.choice([2, 3, 4, 5, 7, 8, 15, 16, 17, 31, 33, 64, tall]))
        batch = int(rng.choice([1, 1, 2, 3, 5]))
        if nx * ny * batch > (4000000 if large else 600000):
            continue
        n = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 9, 12, 13]))
        ratio = float(rng.choice([1.0, 1.0, 0.5, 1.6]))
        wl = workloads.random_problem(int(rng.integers(1 << 30)), nx, ny, batch=batch, dy_ratio=ratio)
        ref = [oracle.step(wl.U[s], wl.V[s], wl.W[s], wl.a, wl.b, wl.c, r=wl.r[s], d=wl.d[s],
                           alpha=wl.alpha[s], c_r=wl.c_r[s], n=n, dt=wl.dt, dx=wl.h, dy=wl.dy)
               for s in range(batch)]
        outs = {}
        for name, k in KERNELS.items():
            try:
                with B.from_workload(wl, dtype=dtype) as sim:
                    sim.set_option(B.GG_OPT_KERNEL, k)
                    if rng.random() < 0.3:
                        sim.set_option(B.GG_OPT_ITEMS_PER_WARP, int(rng.choice([1, 2, 16])))
                    sim.step(n, wl.dt)
                    outs[name] = sim.get_state_numpy()
            except B.GGError as e:
                if e.code != B.GG_ERR_UNSUPPORTED:      # a shape the kernel declares it cannot take
                    raise
        tol = 1e-10 if dtype == "f64" else 2e-4
        for name, got in outs.items():
            err = max(float(np.max(np.abs(got[f][s].astype(np.float64) - ref[s][f])))
                      for f in range(3) for s in range(batch))
            same = all(np.array_equal(got[f], outs["generic"][f]) for f in range(3))
            if not (err <= tol) or not same:
                bad += 1
                print("BAD", dtype, nx, ny, batch, n, ratio, name, err, same, flush=True)
        ncase += 1
    print(f"fuzz: {ncase} cases, {bad} bad", flush=True)
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
