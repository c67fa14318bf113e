"""Full-length, WHOLE-FIELD parity of BASELINE.json's configs 2, 3 and 4 (-m gpu): the stated grid,
the stated step count, AUTO kernel selection with graphs on (what bench.py times), every cell of
U, V, W compared with the CPU oracle on the same seeded inputs.  Bars are north_star's: fp64
max-abs <= 1e-10 per field, fp32 storage <= 2e-4.  (Configs 0 and 1 run at full length in
test_gpu_parity.py; this file is named to be collected LAST so that `-x` meets the fast tests
first.  Oracle wall time on the GPU box's 16 host cores: 3 x ~70 s, ~120 s and 16 x ~7 s.)

The step is eq. (3), with Tables 1-2.
"""
import time

import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-10, "f32": 2e-4}


def gpu_final(wl, dtype):
    with binding.from_workload(wl, dtype=dtype) as sim:
        kernel = sim.kernel
        sim.step(wl.steps, wl.dt)
        ms = sim.last_step_ms()
        out = sim.get_state_numpy()
    return out, kernel, ms


def oracle_final(wl, s):
    t0 = time.perf_counter()
    ref = oracle.step(wl.U[s], wl.V[s], wl.W[s], wl.a, wl.b, wl.c, r=wl.r[s], d=wl.d[s],
                      alpha=wl.alpha[s], c_r=wl.c_r[s], n=wl.steps, dt=wl.dt, dx=wl.h)
    return ref, time.perf_counter() - t0


def compare(got, ref, s, dtype, what):
    errs = [float(np.max(np.abs(got[f][s].astype(np.float64) - ref[f]))) for f in range(3)]
    print(f"{what}: max-abs err U,V,W = {errs[0]:.2e} {errs[1]:.2e} {errs[2]:.2e} (bar {TOL[dtype]:g})")
    assert max(errs) <= TOL[dtype], (what, errs)
    return errs


@pytest.mark.parametrize("d", [2.0, 10.0, 20.0])
def test_config2_full_length_whole_field(d):
    """2048^2, smooth heterogeneous tensor, 10^4 steps, at EVERY d of the sweep {2, 10, 20}
    (BASELINE.json configs[2]; the aggressiveness d decides whether an interstitial
    gap forms, so the three runs stress the reaction term d U W of eq. (1) very differently over
    10^4 steps).  Same inputs, same dt; only d changes."""
    wl = workloads.make(2, d=d)
    assert (wl.nx, wl.ny, wl.steps) == (2048, 2048, 10000) and wl.d[0] == d
    got, kernel, ms = gpu_final(wl, "f64")
    assert kernel == "quad"
    ref, osec = oracle_final(wl, 0)
    compare(got, ref, 0, "f64", f"cfg2 d={d:g} {kernel} gpu {ms:.0f} ms oracle {osec:.0f} s")
    # the run is not trivial: W started at 0 everywhere and the seeded noise on V has grown the
    # tumour (and its acid) over the whole dish by t = n dt
    assert np.max(np.abs(ref[2] - wl.W[0])) > 0.5 and np.max(np.abs(ref[1] - wl.V[0])) > 0.5


def test_config3_full_length_whole_field_both_dtypes():
    """8192^2, layered discontinuous tensor, 1000 steps, fp64 AND fp32 storage against ONE oracle
    run (the oracle always computes in fp64 from the fp64 inputs, reading A10)."""
    wl = workloads.make(3)
    assert (wl.nx, wl.ny, wl.steps) == (8192, 8192, 1000)
    got64, k64, ms64 = gpu_final(wl, "f64")
    got32, k32, ms32 = gpu_final(wl, "f32")
    assert k64 == "quad" and k32 in ("pair", "quad")
    ref, osec = oracle_final(wl, 0)
    compare(got64, ref, 0, "f64", f"cfg3 f64 {k64} gpu {ms64:.0f} ms oracle {osec:.0f} s")
    compare(got32, ref, 0, "f32", f"cfg3 f32 {k32} gpu {ms32:.0f} ms")


CFG4_SIMS = sorted(set(range(0, 64, 4)) | {1, 31, 62, 63})   # 20 of the 64: every 4th (32 among them) + both ends + the middle


def test_config4_full_length_whole_field_twenty_simulations():
    """64 x 1024^2 in one batch, 5000 steps.  Twenty simulations are compared whole-field, each
    against its own independent oracle run: every fourth one (so every region of the log-spaced d
    sweep 0.5 .. 20 with alpha = 1e-4), the alpha = 1e-3 partners at both ends and in the middle
    (1, 31, 63) and 62.  (All 64 would add ~5 min of oracle time to the GPU tier; DESIGN.md
    section 6 states the choice.)"""
    wl = workloads.make(4)
    assert (wl.batch, wl.nx, wl.ny, wl.steps) == (64, 1024, 1024, 5000)
    got, kernel, ms = gpu_final(wl, "f64")
    assert kernel == "quad"
    assert len(CFG4_SIMS) == 20
    for s in CFG4_SIMS:
        ref, osec = oracle_final(wl, s)
        compare(got, ref, s, "f64", f"cfg4 sim {s} d={wl.d[s]:.3g} alpha={wl.alpha[s]:g} oracle {osec:.0f} s")
    assert np.max(np.abs(got[0][0] - got[0][62])) > 1e-3   # the sweep's ends really differ
