#!/usr/bin/env python
"""One resident-kernel call on a small grid (for ncu captures of gg_step_resident; bench.py times
the 8192^2 headline workload, which never runs this kernel).

    python tests/resident_probe.py [cfg] [dtype] [steps]      # default: 1 f32 64 (512^2)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from paper_2006_01748_b200 import binding, workloads  # noqa: E402

cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 1
dtype = sys.argv[2] if len(sys.argv) > 2 else "f32"
steps = int(sys.argv[3]) if len(sys.argv) > 3 else 64
wl = workloads.make(cfg)
with binding.from_workload(wl, dtype=dtype) as sim:
    sim.set_option(binding.GG_OPT_KERNEL, binding.GG_KERNEL_RESIDENT)
    sim.step(steps, wl.dt)
    ms = sim.last_step_ms()
    got = sim.get_state_numpy()
ref = oracle.step(wl.U[0], wl.V[0], wl.W[0], wl.a, wl.b, wl.c, r=wl.r[0], d=wl.d[0], alpha=wl.alpha[0],
                  c_r=wl.c_r[0], n=steps, dt=wl.dt, dx=wl.h)
err = max(float(np.max(np.abs(g[0].astype(np.float64) - r))) for g, r in zip(got, ref))
print(f"resident {wl.name} {dtype}: {steps} steps in {ms:.3f} ms ({ms / steps * 1e3:.2f} us/step), max-abs err {err:.2e}")
assert err <= (1e-10 if dtype == "f64" else 2e-4)
