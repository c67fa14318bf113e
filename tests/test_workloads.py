"""The seeded input generators (paper_2006_01748_b200/workloads.py) against the recipe DESIGN.md
section 5 states: shapes, parameter values, positive-definite tensors, states in [0, 1], the dt
rule, seeding.  No oracle, no GPU: pure input construction."""
import numpy as np
import pytest

from paper_2006_01748_b200 import workloads

SMALL = {0: dict(), 1: dict(nx=96, ny=80), 2: dict(nx=128, ny=96), 3: dict(nx=120, ny=96),
         4: dict(nx=64, ny=48, batch=6)}


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_recipe_invariants(cfg):
    wl = workloads.make(cfg, **SMALL[cfg])
    ny, nx = wl.a.shape
    assert (nx, ny) == (wl.nx, wl.ny) and wl.h == 1.0 / 64.0
    assert wl.U.shape == wl.V.shape == wl.W.shape == (wl.batch, ny, nx)
    for x in (wl.a, wl.b, wl.c, wl.U, wl.V, wl.W):
        assert x.dtype == np.float64 and np.isfinite(x).all()
    # eq. (2): symmetric positive definite at every cell
    assert (wl.a > 0).all() and (wl.c > 0).all() and (wl.a * wl.c - wl.b ** 2 > 0).all()
    # states: indicator + noise in [0, 1e-3), clipped; no acid initially
    assert wl.U.min() >= 0 and wl.U.max() <= 1 and wl.V.min() >= 0 and wl.V.max() <= 1
    assert not wl.W.any()
    assert ((wl.V > 0.5) == (wl.U < 0.5)).all()          # tumour seed replaces healthy tissue
    assert (wl.V > 0.5).any() and (wl.U > 0.5).any()
    # scalars: r = c_r = 1 everywhere
    assert (wl.r == 1.0).all() and (wl.c_r == 1.0).all()
    # dt = 0.2 h^2 / max(alpha, lambda_max(A))
    lam = float(np.max(0.5 * (wl.a + wl.c) + np.sqrt(0.25 * (wl.a - wl.c) ** 2 + wl.b ** 2)))
    assert wl.dt == pytest.approx(0.2 * wl.h ** 2 / max(float(wl.alpha.max()), lam), rel=1e-14)
    # seeding: the same call gives the same arrays, bit for bit
    again = workloads.make(cfg, **SMALL[cfg])
    for k in ("a", "b", "c", "U", "V"):
        assert np.array_equal(getattr(wl, k), getattr(again, k))


def test_config_specifics():
    w0 = workloads.make(0)
    assert (w0.nx, w0.ny, w0.steps) == (64, 64, 200) and not w0.b.any()
    assert (w0.a == 1e-2).all() and (w0.c == 1e-2).all() and w0.d[0] == 10.0 and w0.alpha[0] == 1e-3
    w1 = workloads.make(1, nx=64, ny=64)
    assert (w1.a == 1.5e-2).all() and (w1.c == 5e-3).all() and (w1.b == 4e-3).all() and w1.steps == 2000
    w2 = workloads.make(2, nx=128, ny=128)
    assert np.abs(w2.a / 1e-2 - 1).max() <= 0.5 + 1e-12 and np.abs(w2.c / 1e-2 - 1).max() <= 0.5 + 1e-12
    assert (np.abs(w2.b) <= 0.8 * np.sqrt(w2.a * w2.c) + 1e-18).all() and w2.steps == 10000
    assert workloads.make(2, nx=64, ny=64, d=20.0).d[0] == 20.0
    w3 = workloads.make(3, nx=96, ny=96)
    assert w3.dtypes == ("f64", "f32") and w3.steps == 1000
    bands = {tuple(row) for row in np.stack([w3.a[:, 0], w3.b[:, 0], w3.c[:, 0]], 1)}
    assert len(bands) == 6 and (w3.a == w3.a[:, :1]).all()          # 6 horizontal bands, constant in x
    assert ((5e-3 <= w3.a) & (w3.a <= 2e-2)).all() and (np.abs(w3.b) <= 0.9 * np.sqrt(w3.a * w3.c)).all()
    w4 = workloads.make(4, nx=64, ny=64)
    assert w4.batch == 64 and w4.steps == 5000
    assert w4.d[0] == pytest.approx(0.5) and w4.d[-1] == pytest.approx(20.0)
    assert (w4.d[0::2] == w4.d[1::2]).all() and (w4.alpha[0::2] == 1e-4).all() and (w4.alpha[1::2] == 1e-3).all()
    assert not np.array_equal(w4.U[0], w4.U[1])                      # noise is drawn per simulation


def test_random_problem_is_positive_definite_and_mesh_ratio():
    wl = workloads.random_problem(1, 40, 30, batch=3, dy_ratio=0.5)
    assert (wl.a * wl.c - wl.b ** 2 > 0).all() and wl.dy == wl.h * 0.5
    assert wl.U.min() >= 0 and wl.U.max() <= 1 and workloads.random_problem(1, 40, 30).hy is None
