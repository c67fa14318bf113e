"""GPU tests (-m gpu) of the device-side reductions next to the step: gg_diagnostics (NEXT-1) and
gg_max_stable_dt (NEXT-2), through the C ABI, against oracle.diagnostics / oracle.lambda_max.

Counts, minima and maxima are decided on the same stored values on both sides (the oracle is fed
the GPU's own state, converted exactly to fp64), so they must agree exactly; the sums differ only
in summation order (both accumulate in fp64): 1e-12 relative.  End to end (GPU state after n steps
vs the oracle's own n steps) the sums agree to the parity tolerance times the cell count.
"""
import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu


def check_diag(got, ref):
    np.testing.assert_allclose(got[:3], ref[:3], rtol=1e-12, atol=1e-12)
    assert list(got[3:]) == list(ref[3:])


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_diagnostics_of_the_gpu_state(dtype):
    wl = workloads.make(4, nx=264, ny=190, batch=5, steps=150)
    with binding.from_workload(wl, dtype=dtype) as sim:
        for eps in (1e-2, 0.3):
            got = sim.diagnostics(eps)
            U, V, W = sim.get_state_numpy()
            for s in range(wl.batch):
                check_diag(got[s], oracle.diagnostics(U[s], V[s], W[s], eps))
        sim.step(wl.steps, wl.dt)
        got = sim.diagnostics(0.3)
        U, V, W = sim.get_state_numpy()
        for s in range(wl.batch):
            check_diag(got[s], oracle.diagnostics(U[s], V[s], W[s], 0.3))
        assert not np.array_equal(got[0], got[-1])      # different d: different diagnostics


def test_diagnostics_end_to_end_against_oracle_steps():
    wl = workloads.make(1, nx=200, ny=120, steps=300)     # b != 0: W undershoots 0, U overshoots 1
    with binding.from_workload(wl) as sim:
        sim.step(wl.steps, wl.dt)
        got = sim.diagnostics(0.05)[0]
    ref_state = oracle.step(wl.U[0], wl.V[0], wl.W[0], wl.a, wl.b, wl.c, r=wl.r[0], d=wl.d[0],
                            alpha=wl.alpha[0], c_r=wl.c_r[0], n=wl.steps, dt=wl.dt, dx=wl.h)
    ref = oracle.diagnostics(*ref_state, 0.05)
    n = wl.nx * wl.ny
    np.testing.assert_allclose(got[:3], ref[:3], rtol=0, atol=1e-10 * n)
    np.testing.assert_allclose(got[5:], ref[5:], rtol=0, atol=1e-10)
    assert abs(got[3] - ref[3]) <= 2 and abs(got[4] - ref[4]) <= 2   # threshold cells may flip


def test_diagnostics_show_the_documented_undershoot():
    """Reading A7: with b != 0 the scheme undershoots W < 0 in the first steps (and nothing clamps
    it); gg_diagnostics reports it exactly as the oracle's state has it."""
    wl = workloads.make(1, nx=200, ny=120, steps=8)
    with binding.from_workload(wl) as sim:
        sim.step(wl.steps, wl.dt)
        got = sim.diagnostics(0.05)[0]
    ref_state = oracle.step(wl.U[0], wl.V[0], wl.W[0], wl.a, wl.b, wl.c, r=wl.r[0], d=wl.d[0],
                            alpha=wl.alpha[0], c_r=wl.c_r[0], n=wl.steps, dt=wl.dt, dx=wl.h)
    ref = oracle.diagnostics(*ref_state, 0.05)
    assert ref[5] < -1e-6 and got[5] < -1e-6
    np.testing.assert_allclose(got[5:], ref[5:], rtol=0, atol=1e-10)


def test_diagnostics_large_grid_many_blocks_and_tail():
    wl = workloads.make(3, nx=2056, ny=1031)              # > 296 segments' worth, ragged tail
    with binding.from_workload(wl) as sim:
        got = sim.diagnostics(1e-2)[0]
    check_diag(got, oracle.diagnostics(wl.U[0], wl.V[0], wl.W[0], 1e-2))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_max_stable_dt(dtype):
    for cfg, kw in ((1, dict(nx=128, ny=96)), (2, dict(nx=520, ny=300)), (3, dict(nx=264, ny=150))):
        wl = workloads.make(cfg, **kw)
        a, b, c = wl.a, wl.b, wl.c
        if dtype == "f32":                                # the GPU sees the rounded tensor
            a, b, c = (x.astype(np.float32).astype(np.float64) for x in (a, b, c))
        with binding.from_workload(wl, dtype=dtype) as sim:
            dt, lam = sim.max_stable_dt(0.2)
        assert abs(lam - oracle.lambda_max(a, b, c)) <= 1e-15
        assert abs(dt - oracle.max_stable_dt(a, b, c, wl.alpha, wl.h, safety=0.2)) <= 1e-15
        if dtype == "f64":
            assert abs(dt - wl.dt) <= 1e-15               # the rule the workloads were built with


def test_max_stable_dt_rectangular_mesh_and_alpha_dominated():
    wl = workloads.random_problem(9, 64, 40, batch=3, dy_ratio=0.5)
    with binding.from_workload(wl) as sim:
        dt, lam = sim.max_stable_dt(0.25)
    assert abs(dt - oracle.max_stable_dt(wl.a, wl.b, wl.c, wl.alpha, wl.h, wl.dy, safety=0.25)) <= 1e-15
    with binding.Simulation(32, 32, 0.5, 1.0, 10.0, 7.0, 1.0) as sim:   # alpha = 7 >> tensor
        sim.set_tensor(np.full((32, 32), 1e-2), np.zeros((32, 32)), np.full((32, 32), 1e-2))
        dt, lam = sim.max_stable_dt(0.2)
    assert lam == 1e-2 and dt == 0.2 * 0.25 / 7.0


def test_reduction_call_order_errors():
    ctx = binding.gg_create(16, 16, 0.5, 1.0, 10.0, 1e-3, 1.0)
    try:
        with pytest.raises(binding.GGError) as e:
            binding.gg_diagnostics(ctx, 1e-2, 1)
        assert e.value.code == binding.GG_ERR_STATE
        with pytest.raises(binding.GGError) as e:
            binding.gg_max_stable_dt(ctx, 0.2)
        assert e.value.code == binding.GG_ERR_STATE
    finally:
        binding.gg_destroy(ctx)
    wl = workloads.make(0)
    with binding.from_workload(wl) as sim:
        for bad in (-1.0, float("nan")):
            with pytest.raises(binding.GGError) as e:
                sim.diagnostics(bad)
            assert e.value.code == binding.GG_ERR_ARG
        with pytest.raises(binding.GGError):
            sim.max_stable_dt(0.0)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_front_positions(dtype):
    wl = workloads.make(4, nx=264, ny=190, batch=4, steps=200)
    with binding.from_workload(wl, dtype=dtype) as sim:
        sim.step(wl.steps, wl.dt)
        U, V, W = sim.get_state_numpy()
        fields = {"U": U, "V": V, "W": W}
        for field, level in (("V", 0.5), ("W", 0.2), ("U", 0.9), ("V", 2.0)):
            for axis, index in ((0, 0), (0, 114), (0, 189), (1, 0), (1, 92), (1, 263)):
                got = sim.front(field, axis, index, level)
                for s in range(wl.batch):
                    assert tuple(got[s]) == oracle.front(fields[field][s], axis, index, level)
        with pytest.raises(binding.GGError) as e:
            sim.front("V", 0, 190, 0.5)
        assert e.value.code == binding.GG_ERR_ARG
        with pytest.raises(binding.GGError):
            sim.front(3, 0, 0, 0.5)


def test_diagnostics_count_nonfinite_cells():
    """Nothing in the step repairs a NaN (eq. (3) has no such rule); gg_diagnostics reports how
    many cells hold one: the extrema skip NaNs (fmin / fmax), the sums do not."""
    wl = workloads.random_problem(12, 200, 90, batch=2)
    U, V, W = wl.U.copy(), wl.V.copy(), wl.W.copy()
    W[1, 40, 17] = np.nan
    U[1, 3, 199] = np.inf
    V[1, 3, 199] = -np.inf          # same cell: counted once
    with binding.from_workload(wl) as sim:
        sim.set_state(U, V, W)
        got = sim.diagnostics(1e-2)
        ref = [oracle.diagnostics(U[s], V[s], W[s], 1e-2) for s in range(2)]
        assert got[0][8] == 0 and got[1][8] == 2
        check_diag(got[0], ref[0])
        assert np.isnan(got[1][2]) and got[1][0] == np.inf and got[1][1] == -np.inf
        assert list(got[1][3:]) == list(ref[1][3:])
        sim.step(4, wl.dt)          # the NaN spreads one cell per step through W's nine-point stencil
        after = sim.diagnostics(1e-2)
        assert after[0][8] == 0 and after[1][8] > 2
