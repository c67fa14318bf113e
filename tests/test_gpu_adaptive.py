"""GPU tests (-m gpu) of the device-resident step size:
dt is never a kernel argument, so graphs survive any dt; gg_step_adaptive re-evaluates dt_k on
the device with no host round trip and matches the oracle's time loop."""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-10, "f32": 2e-4}
KERNELS = {"generic": binding.GG_KERNEL_GENERIC, "stream": binding.GG_KERNEL_STREAM,
           "stream2": binding.GG_KERNEL_STREAM2, "pair": binding.GG_KERNEL_PAIR,
           "quad": binding.GG_KERNEL_QUAD}


def adaptive_problem(seed, nx, ny, batch, alpha):
    """A problem on which the rule really moves dt: alpha (1 - U) above lambda_max(A), U starting
    in [0.6, 1] and decaying under a strong acid term, so the V diffusivity bound grows in time."""
    w = workloads.random_problem(seed, nx, ny, batch=batch)
    return dataclasses.replace(w, U=0.6 + 0.4 * w.U, d=4.0 * w.d,
                               alpha=np.broadcast_to(np.asarray(alpha, dtype=np.float64), (batch,)).copy())


def oracle_adaptive(w, n, safety, every_k):
    return oracle.step_adaptive(w.U, w.V, w.W, w.a, w.b, w.c, r=w.r, d=w.d, alpha=w.alpha, c_r=w.c_r,
                                n=n, safety=safety, every_k=every_k, dx=w.h, dy=w.dy)


def check(got, ref, dtype, what):
    for name, g, r in zip("UVW", got, ref):
        err = float(np.max(np.abs(g.astype(np.float64) - r)))
        assert err <= TOL[dtype], f"{what}: field {name} max-abs error {err:.3e}"


def test_thousand_distinct_dt_capture_each_graph_shape_once():
    """The paper's host loop hands a new dt to every iteration.  1000 gg_step calls
    with 1000 distinct dt values must replay ONE captured graph per (length, parity) -- dt is not
    part of the graph -- and still match the oracle fed with the same sequence of step sizes."""
    wl = workloads.make(3, nx=480, ny=96, steps=8)
    with binding.from_workload(wl) as sim:
        sim.set_option(binding.GG_OPT_KERNEL, binding.GG_KERNEL_QUAD)
        U, V, W = wl.U[0], wl.V[0], wl.W[0]
        for i in range(1000):
            dt = wl.dt * (1.0 - 5e-4 * i)
            sim.step(8, dt)
            U, V, W = oracle.step(U, V, W, wl.a, wl.b, wl.c, r=wl.r[0], d=wl.d[0], alpha=wl.alpha[0],
                                  c_r=wl.c_r[0], n=8, dt=dt, dx=wl.h)
        assert sim.graph_captures == 1, sim.graph_captures
        assert sim.launches == 2000
        t, dt_last, steps = sim.clock()
        assert steps == 8000 and dt_last == wl.dt * (1.0 - 5e-4 * 999)
        assert t == pytest.approx(8 * sum(wl.dt * (1.0 - 5e-4 * i) for i in range(1000)), rel=1e-12)
        got = sim.get_state_numpy()
    check(got, (U[None], V[None], W[None]), "f64", "1000 distinct dt")


@pytest.mark.parametrize("kernel", [None, "generic", "stream", "stream2", "pair", "quad"])
def test_adaptive_parity_every_kernel(kernel):
    w = adaptive_problem(61, 480, 70, 2, [0.2, 0.3])
    n, every_k = 23, 5
    U, V, W, t, dts = oracle_adaptive(w, n, 0.2, every_k)
    assert dts[0] > dts[-1] * 1.01          # the rule really moved dt
    with binding.from_workload(w) as sim:
        if kernel:
            sim.set_option(binding.GG_OPT_KERNEL, KERNELS[kernel])
        sim.step_adaptive(n, 0.2, every_k)
        tg, dtg, steps = sim.clock()
        got = sim.get_state_numpy()
    assert steps == n
    # the reductions are exact, so dt_k is an exact function of the stored U^k -- which agrees
    # with the oracle's U^k to rounding only (FMA contraction, flux form): compare to 1e-12
    assert dtg == pytest.approx(dts[-1], rel=1e-12)
    assert tg == pytest.approx(t, rel=1e-12)
    check(got, (U, V, W), "f64", f"adaptive {kernel}")


def test_adaptive_fp32_storage():
    w = adaptive_problem(62, 512, 64, 1, [0.25])
    U, V, W, t, dts = oracle_adaptive(w, 40, 0.2, 4)
    with binding.from_workload(w, dtype="f32") as sim:
        sim.step_adaptive(40, 0.2, 4)
        tg, dtg, steps = sim.clock()
        got = sim.get_state_numpy()
    assert steps == 40 and dtg == pytest.approx(dts[-1], rel=1e-5) and tg == pytest.approx(t, rel=1e-5)
    check(got, (U, V, W), "f32", "adaptive fp32")


def test_adaptive_headline_kernel_graphs_survive_safety_and_match_plain_launches():
    """A grid on which AUTO runs the four-step kernel; every_k = 4 (one launch per dt_k).  A second
    call with another safety factor replays the same graphs; graphs off gives the same bits."""
    w = adaptive_problem(63, 1024, 256, 1, [0.3])
    U, V, W, t1, d1 = oracle_adaptive(w, 64, 0.2, 4)
    w2 = dataclasses.replace(w, U=U, V=V, W=W)
    U2, V2, W2, t2, d2 = oracle_adaptive(w2, 64, 0.1, 4)
    outs = []
    for graph in (1, 0):
        with binding.from_workload(w) as sim:
            assert sim.kernel == "quad"
            sim.set_option(binding.GG_OPT_GRAPH, graph)
            sim.step_adaptive(64, 0.2, 4)
            caps = sim.graph_captures
            sim.step_adaptive(64, 0.1, 4)
            assert sim.graph_captures == caps == (1 if graph else 0)
            assert sim.launches == 32
            tg, dtg, steps = sim.clock()
            outs.append(sim.get_state_numpy())
        assert steps == 128 and dtg == pytest.approx(d2[-1], rel=1e-12) and tg == pytest.approx(t1 + t2, rel=1e-12)
        check(outs[-1], (U2[None], V2[None], W2[None]), "f64", f"adaptive quad graph={graph}")
    assert all(np.array_equal(x, y) for x, y in zip(*outs))


def test_adaptive_small_grid_and_resident_refusal():
    w = adaptive_problem(64, 64, 48, 1, [0.3])
    U, V, W, t, dts = oracle_adaptive(w, 17, 0.2, 3)
    with binding.from_workload(w) as sim:
        assert sim.kernel == "resident"      # AUTO would keep this grid on chip for gg_step ...
        sim.step_adaptive(17, 0.2, 3)        # ... but dt_k needs a launch boundary: STREAM2 runs
        got = sim.get_state_numpy()
        sim.set_option(binding.GG_OPT_KERNEL, binding.GG_KERNEL_RESIDENT)
        with pytest.raises(binding.GGError) as e:
            sim.step_adaptive(4, 0.2, 2)
        assert e.value.code == binding.GG_ERR_UNSUPPORTED
    check(got, (U[None], V[None], W[None]), "f64", "adaptive small")


def test_first_adaptive_dt_is_bit_identical_to_the_oracle_rule():
    """Before any step the stored state IS the oracle's: the device-side rule (exact max / min
    reductions, the same three roundings) must give the oracle's dt_0 bit for bit."""
    w = adaptive_problem(65, 236, 33, 3, [0.2, 0.05, 0.3])
    want = oracle.adaptive_dt(w.U, w.a, w.b, w.c, w.alpha, w.h, safety=0.17)
    with binding.from_workload(w) as sim:
        sim.step_adaptive(1, 0.17, 1)
        t, dt, steps = sim.clock()
    assert steps == 1 and dt == want and t == want


def test_clock_counts_fixed_steps_and_resets_on_set_state():
    wl = workloads.make(0)
    with binding.from_workload(wl) as sim:
        sim.step(10, wl.dt)
        sim.step(3, 0.5 * wl.dt)
        t, dt, steps = sim.clock()
        assert steps == 13 and dt == 0.5 * wl.dt and t == pytest.approx(11.5 * wl.dt, rel=1e-15)
        sim.set_state(wl.U, wl.V, wl.W)
        assert sim.clock()[0] == 0.0 and sim.clock()[2] == 0
        with pytest.raises(binding.GGError):
            sim.step_adaptive(4, 0.0, 1)
        with pytest.raises(binding.GGError):
            sim.step_adaptive(4, 0.2, 0)


def test_adaptive_rule_without_a_bound_freezes_the_state_and_is_reported():
    """A zero tensor with alpha = 0 leaves the rule dt = safety h^2 / max(lambda_max, alpha (1 - min U))
    without a positive denominator.  The device must not fold inf or NaN into the step: those steps
    run with dt = 0 (state and simulated time untouched), gg_get_clock reports GG_ERR_ARG, further
    step calls are refused, and gg_set_state puts the context back to work."""
    w = adaptive_problem(66, 96, 40, 2, [0.0, 0.0])
    zero = np.zeros_like(w.a)
    with binding.from_workload(w) as sim:
        sim.set_tensor(zero, zero, zero)
        before = sim.get_state_numpy()
        sim.step_adaptive(6, 0.2, 2)                    # enqueues: the failure shows on the device
        after = sim.get_state_numpy()
        for b, a in zip(before, after):
            assert np.array_equal(b, a)
        with pytest.raises(binding.GGError) as e:
            sim.clock()
        assert e.value.code == binding.GG_ERR_ARG and "no positive finite bound in 3 evaluation" in str(e.value)
        for call in (lambda: sim.step(1, 1e-3), lambda: sim.step_adaptive(1, 0.2, 1)):
            with pytest.raises(binding.GGError) as e:
                call()
            assert e.value.code == binding.GG_ERR_ARG
        sim.set_state(w.U, w.V, w.W)                    # clears the flag on both sides
        assert sim.clock()[0] == 0.0 and sim.clock()[2] == 0
        sim.step(2, 1e-3)
        t, dt, steps = sim.clock()
        assert steps == 2 and dt == 1e-3 and t == pytest.approx(2e-3, rel=1e-15)
        assert not np.array_equal(sim.get_state_numpy()[0], before[0])


def test_two_live_contexts_of_different_shapes_share_kernels():
    """The opt-in shared-memory limit is a per-FUNCTION attribute: a second context with a smaller
    shape must not lower it under a first context's feet (resident and pair instantiations)."""
    big = workloads.make(3, nx=512, ny=512, steps=16)
    small = workloads.make(3, nx=64, ny=64, steps=16)
    ref_big = oracle.step(big.U[0], big.V[0], big.W[0], big.a, big.b, big.c, r=1.0, d=10.0, alpha=1e-3,
                          c_r=1.0, n=32, dt=big.dt, dx=big.h)
    for kernel, dtype in ((binding.GG_KERNEL_RESIDENT, "f32"), (binding.GG_KERNEL_PAIR, "f64"),
                          (binding.GG_KERNEL_QUAD, "f64")):
        with binding.from_workload(big, dtype=dtype) as s1, binding.from_workload(small, dtype=dtype) as s2:
            s1.set_option(binding.GG_OPT_KERNEL, kernel)
            s2.set_option(binding.GG_OPT_KERNEL, kernel)
            s1.step(16, big.dt)          # plan of the large shape ...
            s2.step(16, small.dt)        # ... then the small one (used to lower the attribute)
            s1.step(16, big.dt)          # the large shape must still launch
            got = s1.get_state_numpy()
        check(got, tuple(r[None] for r in ref_big), dtype, f"two contexts, kernel {kernel}")
