"""Pins for the CPU oracle (oracle/gg_oracle.cpp) against what the paper and the mathematics fix.

None of these re-types the oracle's own formula: they are hand-computed values (tests/golden),
closed forms of the printed stencils, special cases that reduce to independent textbook codes
(scalar ODE recursion, 1-D scheme), invariants (conservation, symmetries, equilibria, bounds), a
many-step discrete-cosine eigenmode solution, and a brute-force evaluation of Tables 1-2 *as
printed* (entry times value, with the printed centre entries) in pure Python on tiny grids.
Citations: PAPER.md:74 (eq. 3), :81-85 (Table 1), :89-92 (Table 2), :42/:77 (Neumann).
"""
import math

import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import workloads


def XY(n=4):
    X = np.arange(1, n + 1, dtype=np.float64)[None, :] * np.ones((n, 1))
    Y = np.arange(1, n + 1, dtype=np.float64)[:, None] * np.ones((1, n))
    return X, Y


# ---------------------------------------------------------------------------------------------
# 7. hand-computed 4x4 values (P1, P2, P3, P5)
# ---------------------------------------------------------------------------------------------
def test_P1_D2_constant_tensor(golden):
    X, Y = XY()
    W = X * X + X * Y
    a, b, c = np.full_like(W, 2.0), np.full_like(W, 1.0), np.full_like(W, 3.0)
    got = oracle.D2(a, b, c, W, 1.0, 1.0)
    np.testing.assert_allclose(got, golden("p1_D2_const_tensor.txt"), rtol=0, atol=1e-12)
    assert abs(got.sum()) < 1e-12  # zero-flux boundaries: the operator sums to zero
    # the rejected reading A' (b even) would give 11.5 at (0,0) and a total of 18
    assert abs(got[0, 0] - 14.0) < 1e-12


def test_P2_D2_heterogeneous_tensor(golden):
    X, Y = XY()
    W = X * X + X * Y
    a, b, c = 1 + 0.25 * X, 0.5 + 0.25 * (X - Y), 2 + 0.5 * Y
    got = oracle.D2(a, b, c, W, 1.0, 1.0)
    np.testing.assert_allclose(got, golden("p2_D2_hetero_tensor.txt"), rtol=0, atol=1e-12)
    assert abs(got.sum()) < 1e-12


def test_P3_D1(golden):
    X, Y = XY()
    U = 0.1 * X + 0.05 * Y
    V = X * X + Y * Y
    got = oracle.D1(U, V, 1.0, 1.0)
    np.testing.assert_allclose(got, golden("p3_D1.txt"), rtol=0, atol=1e-12)
    assert abs(got.sum()) < 1e-12


def test_P5_full_step(golden):
    X, Y = XY()
    U0 = 0.1 * X + 0.05 * Y
    V0 = 0.02 * (X * X + Y * Y)
    W0 = 0.01 * (X * X + X * Y)
    a, b, c = 1 + 0.25 * X, 0.5 + 0.25 * (X - Y), 2 + 0.5 * Y
    U1, V1, W1 = oracle.step(U0, V0, W0, a, b, c, r=1.0, d=10.0, alpha=0.5, c_r=2.0, n=1,
                             dt=0.01, dx=0.5)
    np.testing.assert_allclose(U1, golden("p5_step_U1.txt"), rtol=0, atol=1e-12)
    np.testing.assert_allclose(V1, golden("p5_step_V1.txt"), rtol=0, atol=1e-12)
    np.testing.assert_allclose(W1, golden("p5_step_W1.txt"), rtol=0, atol=1e-12)
    # the one cell worked by hand in the fixture header
    assert abs(U1[0, 0] - (0.15 + 0.01 * 0.15 * 0.85 - 10 * 0.01 * 0.15 * 0.02)) < 1e-15


# ---------------------------------------------------------------------------------------------
# brute force: Tables 1 and 2 exactly as printed (entry x value, printed centre entries), tiny grids
# ---------------------------------------------------------------------------------------------
def _ghost(P, i, j, odd=False):
    """Pure-Python mirrored read P[j][i] with i in [-1,nx], j in [-1,ny] (reading A2/A12)."""
    ny, nx = len(P), len(P[0])
    s = 1.0
    ii, jj = i, j
    if i < 0:
        ii, s = 0, -s
    if i >= nx:
        ii, s = nx - 1, -s
    if j < 0:
        jj, s = 0, -s
    if j >= ny:
        jj, s = ny - 1, -s
    return (s if odd else 1.0) * P[jj][ii]


def table2_as_printed(a, b, c, W, dx, dy):
    ny, nx = len(W), len(W[0])
    out = [[0.0] * nx for _ in range(ny)]
    for j in range(ny):
        for i in range(nx):
            A = lambda di, dj: _ghost(a, i + di, j + dj)
            B = lambda di, dj: _ghost(b, i + di, j + dj, odd=True)
            C = lambda di, dj: _ghost(c, i + di, j + dj)
            w = lambda di, dj: _ghost(W, i + di, j + dj)
            ent = {
                (-1, +1): -(B(-1, 0) + B(0, 1)) / (4 * dx * dy),
                (0, +1): (C(0, 0) + C(0, 1)) / (2 * dy * dy),
                (+1, +1): (B(1, 0) + B(0, 1)) / (4 * dx * dy),
                (-1, 0): (A(-1, 0) + A(0, 0)) / (2 * dx * dx),
                (0, 0): -(A(-1, 0) + 2 * A(0, 0) + A(1, 0)) / (2 * dx * dx)
                        - (C(0, -1) + 2 * C(0, 0) + C(0, 1)) / (2 * dy * dy),
                (+1, 0): (A(0, 0) + A(1, 0)) / (2 * dx * dx),
                (-1, -1): (B(-1, 0) + B(0, -1)) / (4 * dx * dy),
                (0, -1): (C(0, -1) + C(0, 0)) / (2 * dy * dy),
                (+1, -1): -(B(1, 0) + B(0, -1)) / (4 * dx * dy),
            }
            out[j][i] = sum(e * w(di, dj) for (di, dj), e in ent.items())
    return np.array(out)


def table1_as_printed(U, V, dx, dy):
    ny, nx = len(U), len(U[0])
    out = [[0.0] * nx for _ in range(ny)]
    for j in range(ny):
        for i in range(nx):
            u = lambda di, dj: _ghost(U, i + di, j + dj)
            v = lambda di, dj: _ghost(V, i + di, j + dj)
            ent = {
                (0, +1): 1 / dy**2 - (u(0, 0) + u(0, 1)) / (2 * dy**2),
                (-1, 0): 1 / dx**2 - (u(-1, 0) + u(0, 0)) / (2 * dx**2),
                # centre entry: printed over two table rows, reading A3
                (0, 0): -2 / dx**2 + (u(-1, 0) + 2 * u(0, 0) + u(1, 0)) / (2 * dx**2)
                        - 2 / dy**2 + (u(0, -1) + 2 * u(0, 0) + u(0, 1)) / (2 * dy**2),
                (+1, 0): 1 / dx**2 - (u(0, 0) + u(1, 0)) / (2 * dx**2),
                (0, -1): 1 / dy**2 - (u(0, -1) + u(0, 0)) / (2 * dy**2),
            }
            out[j][i] = sum(e * v(di, dj) for (di, dj), e in ent.items())
    return np.array(out)


@pytest.mark.parametrize("nx,ny,dx,dy", [(5, 4, 0.5, 0.25), (2, 2, 1.0, 2.0), (3, 6, 0.3, 0.7)])
def test_bruteforce_tables_as_printed(nx, ny, dx, dy):
    rng = np.random.default_rng(7)
    a = rng.uniform(0.5, 2.0, (ny, nx))
    c = rng.uniform(0.5, 2.0, (ny, nx))
    b = rng.uniform(-0.6, 0.6, (ny, nx))
    W = rng.uniform(0, 1, (ny, nx))
    U = rng.uniform(0, 1, (ny, nx))
    V = rng.uniform(0, 1, (ny, nx))
    ref2 = table2_as_printed(a.tolist(), b.tolist(), c.tolist(), W.tolist(), dx, dy)
    ref1 = table1_as_printed(U.tolist(), V.tolist(), dx, dy)
    scale = 4 * 2.0 / min(dx, dy) ** 2
    np.testing.assert_allclose(oracle.D2(a, b, c, W, dx, dy), ref2, rtol=0, atol=1e-13 * scale)
    np.testing.assert_allclose(oracle.D1(U, V, dx, dy), ref1, rtol=0, atol=1e-13 * scale)


# ---------------------------------------------------------------------------------------------
# P4: closed forms at interior cells (exact for the discrete operators, any dx, dy)
# ---------------------------------------------------------------------------------------------
def test_P4_closed_forms_polynomials():
    nx, ny, dx, dy = 9, 8, 0.5, 0.25
    x = (np.arange(nx) * dx)[None, :] * np.ones((ny, 1))
    y = (np.arange(ny) * dy)[:, None] * np.ones((1, nx))
    I = (slice(1, -1), slice(1, -1))
    # constant tensor, quadratic W: D2 = 2 a al + 2 b be + 2 c ga
    a0, b0, c0 = 0.7, 0.2, 0.4
    al, be, ga = 1.3, -0.8, 0.6
    W = al * x * x + be * x * y + ga * y * y
    got = oracle.D2(np.full_like(W, a0), np.full_like(W, b0), np.full_like(W, c0), W, dx, dy)
    np.testing.assert_allclose(got[I], 2 * a0 * al + 2 * b0 * be + 2 * c0 * ga, atol=1e-11)
    # a(x) = x, W = x^2: d_x(x * 2x) = 4x
    got = oracle.D2(x, np.zeros_like(x), np.ones_like(x), x * x, dx, dy)
    np.testing.assert_allclose(got[I], 4 * x[I], atol=1e-11)
    # b(x) = x, W = x y: d_x(b W_y) = 2x, d_y(b W_x) = x  => 3x
    got = oracle.D2(np.ones_like(x), x, np.ones_like(x), x * y, dx, dy)
    np.testing.assert_allclose(got[I], 3 * x[I], atol=1e-11)
    # b(y) = y, W = x y: d_x(b W_y) = y, d_y(b W_x) = 2y  => 3y (checks the y-side corner factors)
    got = oracle.D2(np.ones_like(x), y, np.ones_like(x), x * y, dx, dy)
    np.testing.assert_allclose(got[I], 3 * y[I], atol=1e-11)
    # c(y) = y, W = y^2 => 4y ; checks 1/dy^2
    got = oracle.D2(np.ones_like(x), np.zeros_like(x), y, y * y, dx, dy)
    np.testing.assert_allclose(got[I], 4 * y[I], atol=1e-11)
    # D1: U = u0 + s x, V = x^2 => 2(1-u0) - 4 s x ; and the y analogue
    u0, s = 0.2, 0.05
    got = oracle.D1(u0 + s * x, x * x, dx, dy)
    np.testing.assert_allclose(got[I], 2 * (1 - u0) - 4 * s * x[I], atol=1e-11)
    got = oracle.D1(u0 + s * y, y * y, dx, dy)
    np.testing.assert_allclose(got[I], 2 * (1 - u0) - 4 * s * y[I], atol=1e-11)


def test_P4_plane_wave_symbol():
    """Interior symbol of Table 2 for a constant tensor: sign and factor of the cross term."""
    nx, ny, dx, dy = 12, 10, 0.4, 0.3
    a0, b0, c0 = 0.9, -0.35, 0.5
    thx, thy = 0.7, -1.1
    i = np.arange(nx)[None, :]
    j = np.arange(ny)[:, None]
    W = np.cos(thx * i + thy * j)
    lam = (-(4 * a0 / dx**2) * math.sin(thx / 2) ** 2 - (4 * c0 / dy**2) * math.sin(thy / 2) ** 2
           - (2 * b0 / (dx * dy)) * math.sin(thx) * math.sin(thy))
    got = oracle.D2(np.full_like(W, a0), np.full_like(W, b0), np.full_like(W, c0), W, dx, dy)
    I = (slice(1, -1), slice(1, -1))
    np.testing.assert_allclose(got[I], lam * W[I], atol=1e-12 * abs(lam) * 10)


# ---------------------------------------------------------------------------------------------
# 1. uniform data => scalar ODE recursion of eq. (3)
# ---------------------------------------------------------------------------------------------
def test_uniform_data_follows_scalar_recursion():
    rng = np.random.default_rng(3)
    nx, ny = 7, 5
    a = rng.uniform(0.5, 2.0, (ny, nx))
    c = rng.uniform(0.5, 2.0, (ny, nx))
    b = rng.uniform(-0.4, 0.4, (ny, nx))
    r, d, alpha, c_r, dt, n = 1.3, 4.0, 0.2, 0.7, 1e-3, 300
    u, v, w = 0.8, 0.1, 0.05
    U, V, W = oracle.step(np.full((ny, nx), u), np.full((ny, nx), v), np.full((ny, nx), w), a, b, c,
                          r=r, d=d, alpha=alpha, c_r=c_r, n=n, dt=dt, dx=0.1, dy=0.07)
    for _ in range(n):
        u, v, w = (u + dt * u * (1 - u) - d * dt * u * w, v + r * dt * v * (1 - v),
                   w + c_r * dt * (v - w))
    # D1 = D2 = 0 exactly on uniform data (difference form) => every cell IS the recursion
    assert np.all(U == U[0, 0]) and np.all(V == V[0, 0]) and np.all(W == W[0, 0])
    assert abs(U[0, 0] - u) <= 1e-15 and abs(V[0, 0] - v) <= 1e-15 and abs(W[0, 0] - w) <= 1e-15


def test_logistic_first_order_convergence():
    """v tracks the analytic logistic curve with O(dt) error that halves when dt halves."""
    nx = ny = 3
    one = np.ones((ny, nx))
    v0, r, T = 0.1, 1.0, 2.0
    exact = v0 * math.exp(r * T) / (1 + v0 * (math.exp(r * T) - 1))
    errs = []
    for n in (200, 400, 800):
        _, V, _ = oracle.step(0 * one, v0 * one, 0 * one, one, 0 * one, one, r=r, d=1.0,
                              alpha=1.0, c_r=0.0, n=n, dt=T / n, dx=1.0)
        errs.append(abs(V[1, 1] - exact))
    assert 1.9 < errs[0] / errs[1] < 2.1 and 1.9 < errs[1] / errs[2] < 2.1


# ---------------------------------------------------------------------------------------------
# 2. equilibria
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("state", [(1.0, 0.0, 0.0), (0.0, 1.0, 1.0), (0.0, 0.0, 0.0)])
def test_equilibria_are_fixed_points_bitwise(state):
    w = workloads.random_problem(5, 9, 6)
    u, v, ww = state
    sh = (6, 9)
    U, V, W = oracle.step(np.full(sh, u), np.full(sh, v), np.full(sh, ww), w.a, w.b, w.c,
                          r=1.1, d=7.0, alpha=1e-3, c_r=0.9, n=50, dt=w.dt, dx=w.h)
    assert np.all(U == u) and np.all(V == v) and np.all(W == ww)


def test_coexistence_equilibrium_d_lt_1():
    """(1-d, 1, 1) is stationary for d < 1 (heterogeneous invasion)."""
    w = workloads.random_problem(6, 8, 8)
    d = 0.4
    sh = (8, 8)
    U, V, W = oracle.step(np.full(sh, 1 - d), np.ones(sh), np.ones(sh), w.a, w.b, w.c, r=1.0, d=d,
                          alpha=1e-3, c_r=1.0, n=100, dt=w.dt, dx=w.h)
    assert np.max(np.abs(U - (1 - d))) < 1e-14
    assert np.all(V == 1.0) and np.all(W == 1.0)


# ---------------------------------------------------------------------------------------------
# 3. conservation ("conservativity"): fixes the b-odd ghost reading A2
# ---------------------------------------------------------------------------------------------
def test_conservation_of_W_and_V_mass():
    w = workloads.random_problem(11, 24, 17, bmax=0.9)
    U0, V0, W0 = w.U[0], w.V[0], w.W[0]
    U, V, W = oracle.step(U0, V0, W0, w.a, w.b, w.c, r=0.0, d=3.0, alpha=2e-3, c_r=0.0, n=1000,
                          dt=w.dt, dx=w.h)
    assert abs(W.sum() - W0.sum()) / W0.sum() < 1e-13
    assert abs(V.sum() - V0.sum()) / V0.sum() < 1e-13
    assert np.max(np.abs(W - W0)) > 1e-3  # something did diffuse


# ---------------------------------------------------------------------------------------------
# 4. 1-D reduction (b = 0): every row equals an independent 1-D code
# ---------------------------------------------------------------------------------------------
def _one_d(U, V, W, a, r, d, alpha, c_r, dt, dx, n):
    U, V, W = U.copy(), V.copy(), W.copy()
    for _ in range(n):
        Up = np.concatenate([U[:1], U, U[-1:]])
        Vp = np.concatenate([V[:1], V, V[-1:]])
        Wp = np.concatenate([W[:1], W, W[-1:]])
        ap = np.concatenate([a[:1], a, a[-1:]])
        fV = (1 - 0.5 * (Up[:-1] + Up[1:])) * (Vp[1:] - Vp[:-1])
        fW = 0.5 * (ap[:-1] + ap[1:]) * (Wp[1:] - Wp[:-1])
        Un = U + dt * U * (1 - U) - d * dt * U * W
        Vn = V + r * dt * V * (1 - V) + alpha * dt / dx**2 * (fV[1:] - fV[:-1])
        Wn = W + c_r * dt * (V - W) + dt / dx**2 * (fW[1:] - fW[:-1])
        U, V, W = Un, Vn, Wn
    return U, V, W


@pytest.mark.parametrize("axis", ["x", "y"])
def test_one_dimensional_reduction(axis):
    rng = np.random.default_rng(21)
    n1, n2 = 40, 6
    u = rng.uniform(0, 1, n1)
    v = rng.uniform(0, 1, n1)
    w = rng.uniform(0, 1, n1)
    a1 = rng.uniform(5e-3, 2e-2, n1)
    other = rng.uniform(5e-3, 2e-2, n1)  # the coefficient of the direction with no variation
    r, d, alpha, c_r, dx, n = 1.0, 10.0, 1e-3, 1.0, 1 / 64, 200
    dt = 0.2 * dx * dx / 2e-2
    U1, V1, W1 = _one_d(u, v, w, a1, r, d, alpha, c_r, dt, dx, n)
    if axis == "x":
        ext = lambda q: np.tile(q[None, :], (n2, 1))
        a, c = ext(a1), ext(other)
    else:
        ext = lambda q: np.tile(q[:, None], (1, n2))
        a, c = ext(other), ext(a1)
    U, V, W = oracle.step(ext(u), ext(v), ext(w), a, np.zeros_like(a), c, r=r, d=d, alpha=alpha,
                          c_r=c_r, n=n, dt=dt, dx=dx)
    for got, ref in ((U, U1), (V, V1), (W, W1)):
        np.testing.assert_allclose(got, ext(ref), rtol=0, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# 5. grid symmetries: transpose, flip, 90-degree rotation
# ---------------------------------------------------------------------------------------------
def _run(w, U, V, W, a, b, c, dx, dy, n=25):
    return oracle.step(U, V, W, a, b, c, r=1.0, d=6.0, alpha=1e-3, c_r=1.0, n=n, dt=0.5 * w.dt,
                       dx=dx, dy=dy)


def test_symmetries_transpose_flip_rotate():
    w = workloads.random_problem(31, 13, 9)
    U0, V0, W0 = w.U[0], w.V[0], w.W[0]
    dx, dy = w.h, 1.25 * w.h
    ref = _run(w, U0, V0, W0, w.a, w.b, w.c, dx, dy)
    # (i) transpose: swap i<->j, a<->c, b kept, dx<->dy
    T = lambda q: np.ascontiguousarray(q.T)
    got = _run(w, T(U0), T(V0), T(W0), T(w.c), T(w.b), T(w.a), dy, dx)
    for g, r_ in zip(got, ref):
        np.testing.assert_allclose(T(g), r_, rtol=0, atol=1e-12)
    # (ii) flip in x: reverse i, b -> -b
    F = lambda q: np.ascontiguousarray(q[:, ::-1])
    got = _run(w, F(U0), F(V0), F(W0), F(w.a), -F(w.b), F(w.c), dx, dy)
    for g, r_ in zip(got, ref):
        np.testing.assert_allclose(F(g), r_, rtol=0, atol=1e-12)
    # (iii) 90-degree rotation: rot90 of every array, a<->c, b -> -b, dx<->dy
    R = lambda q: np.ascontiguousarray(np.rot90(q))
    got = _run(w, R(U0), R(V0), R(W0), R(w.c), -R(w.b), R(w.a), dy, dx)
    for g, r_ in zip(got, ref):
        np.testing.assert_allclose(np.rot90(g, -1), r_, rtol=0, atol=1e-12)
    # and the symmetry is not vacuous: without negating b the flipped run differs
    bad = _run(w, F(U0), F(V0), F(W0), F(w.a), F(w.b), F(w.c), dx, dy)
    assert np.max(np.abs(F(bad[2]) - ref[2])) > 1e-6


# ---------------------------------------------------------------------------------------------
# P6: many-step closed form -- discrete cosine eigenmodes of the mirrored grid (b=0, no reactions)
# ---------------------------------------------------------------------------------------------
def test_P6_cosine_eigenmode_many_steps():
    nx, ny, k, l, h = 8, 6, 3, 2, 0.25
    a0, c0 = 0.7, 0.3
    i = np.arange(nx)[None, :]
    j = np.arange(ny)[:, None]
    W0 = np.cos(math.pi * k * (i + 0.5) / nx) * np.cos(math.pi * l * (j + 0.5) / ny)
    lam = (-(4 * a0 / h**2) * math.sin(math.pi * k / (2 * nx)) ** 2
           - (4 * c0 / h**2) * math.sin(math.pi * l / (2 * ny)) ** 2)
    assert abs(lam - (-18.627891115)) < 1e-8  # value quoted in SURVEY.md P6
    dt, n = 0.2 * h * h / a0, 60
    z = np.zeros_like(W0)
    _, _, W = oracle.step(z, z, W0, np.full_like(W0, a0), z, np.full_like(W0, c0), r=0.0, d=0.0,
                          alpha=0.0, c_r=0.0, n=n, dt=dt, dx=h)
    np.testing.assert_allclose(W, (1 + dt * lam) ** n * W0, rtol=0, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# 6. bounds for b = 0 under the step-size bound; documented violation for b != 0
# ---------------------------------------------------------------------------------------------
def test_bounds_hold_for_b_zero_config0():
    w = workloads.make(0)
    U, V, W = w.U[0], w.V[0], w.W[0]
    for _ in range(10):
        U, V, W = oracle.step(U, V, W, w.a, w.b, w.c, r=1.0, d=10.0, alpha=1e-3, c_r=1.0, n=20,
                              dt=w.dt, dx=w.h)
        for F in (U, V, W):
            assert F.min() >= 0.0 and F.max() <= 1.0


def test_bounds_hold_for_b_zero_heterogeneous():
    w = workloads.random_problem(41, 20, 20)
    b = np.zeros_like(w.b)
    dt = 0.2 * w.h**2 / max(w.a.max(), w.c.max())
    U, V, W = w.U[0], w.V[0], w.W[0]
    for _ in range(5):
        U, V, W = oracle.step(U, V, W, w.a, b, w.c, r=1.0, d=10.0, alpha=1e-3, c_r=1.0, n=20,
                              dt=dt, dx=w.h)
        for F in (U, V, W):
            assert F.min() >= 0.0 and F.max() <= 1.0


def test_documented_undershoot_with_cross_term():
    """b != 0: Table 2 has two negative corner weights, so W undershoots 0 (reading A7).  The
    scheme must NOT be 'fixed' by clamping; this asserts the violation exists."""
    w = workloads.make(1, nx=128, steps=8)
    U, V, W = w.U[0], w.V[0], w.W[0]
    wmin, umax = 0.0, 0.0
    for _ in range(8):
        U, V, W = oracle.step(U, V, W, w.a, w.b, w.c, r=1.0, d=10.0, alpha=1e-3, c_r=1.0, n=1,
                              dt=w.dt, dx=w.h)
        wmin, umax = min(wmin, W.min()), max(umax, U.max())
    assert wmin < -5e-5      # W undershoots at the staircase corners of the disk
    assert umax > 1.0 + 1e-6  # and U then overshoots 1


# ---------------------------------------------------------------------------------------------
# host-side facts the configs rely on, and thread-count independence
# ---------------------------------------------------------------------------------------------
def test_dt_rule_values():
    assert abs(workloads.make(0).dt - 4.8828125e-3) < 1e-15
    w1 = workloads.make(1, nx=64, steps=1)
    assert abs(workloads.lambda_max(w1.a, w1.b, w1.c) - 1.6403124237e-2) < 1e-11
    assert abs(w1.dt - 2.9767576160e-3) < 1e-12


def test_thread_count_does_not_change_bits():
    w = workloads.random_problem(51, 33, 29)
    kw = dict(r=1.0, d=9.0, alpha=1e-3, c_r=1.0, n=7, dt=w.dt, dx=w.h)
    r1 = oracle.step(w.U[0], w.V[0], w.W[0], w.a, w.b, w.c, threads=1, **kw)
    r4 = oracle.step(w.U[0], w.V[0], w.W[0], w.a, w.b, w.c, threads=4, **kw)
    for x, y in zip(r1, r4):
        assert np.array_equal(x, y)


def test_bad_arguments_rejected():
    z = np.zeros((1, 5))
    with pytest.raises(ValueError):
        oracle.D1(z, z, 1.0, 1.0)
    z = np.zeros((4, 4))
    with pytest.raises(ValueError):
        oracle.step(z, z, z, z, z, z, r=1, d=1, alpha=1, c_r=1, n=-1, dt=0.1, dx=1.0)


# ---------------------------------------------------------------------------------------------
# Reductions next to the step (NEXT-1 diagnostics, NEXT-2 step bound)
# ---------------------------------------------------------------------------------------------
def test_lambda_max_against_library_eigensolver_and_closed_forms():
    rng = np.random.default_rng(5)
    a = rng.uniform(5e-3, 2e-2, (7, 9))
    c = rng.uniform(5e-3, 2e-2, (7, 9))
    b = rng.uniform(-0.9, 0.9, (7, 9)) * np.sqrt(a * c)
    mats = np.stack([np.stack([a, b], -1), np.stack([b, c], -1)], -2)     # [...,2,2]
    lib = float(np.max(np.linalg.eigvalsh(mats)[..., 1]))                 # LAPACK, not the formula
    assert abs(oracle.lambda_max(a, b, c) - lib) <= 1e-15
    # closed forms: diagonal tensor -> max(a, c); a = c -> a + |b|
    assert oracle.lambda_max(np.full((3, 3), 2.0), np.zeros((3, 3)), np.full((3, 3), 5.0)) == 5.0
    assert abs(oracle.lambda_max(np.full((3, 3), 2.0), np.full((3, 3), -0.5), np.full((3, 3), 2.0)) - 2.5) < 1e-15
    # config 1: lambda_max = 1.6403124237e-2, dt = 2.9767576160e-3
    wl = workloads.make(1, nx=16, ny=16)
    assert abs(oracle.lambda_max(wl.a, wl.b, wl.c) - 1.6403124237e-2) < 1e-11
    assert abs(oracle.max_stable_dt(wl.a, wl.b, wl.c, wl.alpha, wl.h) - 2.9767576160e-3) < 1e-12
    # alpha dominates when the tensor is small; dx != dy takes the smaller mesh size
    assert oracle.max_stable_dt(wl.a * 1e-3, wl.b * 1e-3, wl.c * 1e-3, [1e-3], 0.5, 0.25, safety=0.2) \
        == 0.2 * 0.25 ** 2 / 1e-3


def test_diagnostics_brute_force_and_special_cases():
    rng = np.random.default_rng(6)
    U = rng.uniform(0, 0.05, (5, 7)); V = rng.uniform(0, 1, (5, 7)); W = rng.uniform(-1e-3, 1, (5, 7))
    eps = 0.02
    got = oracle.diagnostics(U, V, W, eps)
    su = sv = sw = 0.0
    gap = tum = 0
    mnw, mxu, mxw = math.inf, -math.inf, -math.inf
    for j in range(5):
        for i in range(7):
            su += U[j, i]; sv += V[j, i]; sw += W[j, i]
            gap += int(U[j, i] < eps and V[j, i] < eps)
            tum += int(V[j, i] >= 0.5)
            mnw = min(mnw, W[j, i]); mxu = max(mxu, U[j, i]); mxw = max(mxw, W[j, i])
    np.testing.assert_allclose(got[:3], [su, sv, sw], rtol=1e-14)
    assert (got[3], got[4], got[5], got[6], got[7], got[8]) == (gap, tum, mnw, mxu, mxw, 0)
    # the healthy state (1,0,0): no gap, no tumour; the invaded state (0,1,1): no gap, all tumour;
    # (0,0,w): every cell is gap
    n = 12
    one, zero = np.ones((3, 4)), np.zeros((3, 4))
    assert list(oracle.diagnostics(one, zero, zero, 1e-2)) == [n, 0, 0, 0, 0, 0, 1, 0, 0]
    assert list(oracle.diagnostics(zero, one, one, 1e-2)) == [0, n, n, 0, n, 1, 0, 1, 0]
    bad = one.copy(); bad[1, 2] = np.nan; bad[0, 0] = np.inf
    d = oracle.diagnostics(zero, bad, bad * 0.5, 1e-2)     # NaN / Inf cells are counted, extrema skip NaN
    assert d[8] == 2 and d[5] == 0.5 and d[7] == np.inf and np.isnan(d[1])
    assert oracle.diagnostics(zero, zero, one * 0.3, 1e-2)[3] == n
    # thresholds are strict / inclusive as documented: U == eps is not gap, V == 1/2 is tumour
    assert oracle.diagnostics(one * 1e-2, zero, zero, 1e-2)[3] == 0
    assert oracle.diagnostics(zero, one * 0.5, zero, 1e-2)[4] == n


def test_gap_opens_for_large_d_only():
    """d > 1 (homogeneous invasion) leaves an interstitial gap between the
    fronts, d < 1 (heterogeneous invasion) does not: normal cells coexist behind the front.
    Noise-free disk data (the configs' V noise seeds tumour growth everywhere)."""
    wl = workloads.make(0)
    inside = wl.V[0] > 0.5
    U0, V0, W0 = np.where(inside, 0.0, 1.0), np.where(inside, 1.0, 0.0), np.zeros(inside.shape)
    gaps = {}
    for d in (0.5, 40.0):
        U, V, W = oracle.step(U0, V0, W0, wl.a, wl.b, wl.c, r=1.0, d=d, alpha=1e-3, c_r=1.0, n=600,
                              dt=wl.dt, dx=wl.h)
        gaps[d] = oracle.diagnostics(U, V, W, 0.2)[3]
    assert gaps[0.5] == 0 and gaps[40.0] > 100


def test_front_positions_brute_force_and_disk():
    rng = np.random.default_rng(7)
    F = rng.uniform(0, 1, (6, 9))
    for axis, n in ((0, 6), (1, 9)):
        for index in range(n):
            line = [F[index][i] for i in range(9)] if axis == 0 else [F[j][index] for j in range(6)]
            hits = [q for q, x in enumerate(line) if x >= 0.6]
            want = (hits[0], hits[-1]) if hits else (-1, -1)
            assert oracle.front(F, axis, index, 0.6) == want
    assert oracle.front(np.zeros((4, 5)), 0, 2, 0.5) == (-1, -1)
    assert oracle.front(np.full((4, 5), 0.5), 1, 3, 0.5) == (0, 3)      # >= is inclusive
    # the seeded disk of config 0 (radius 6.4 cells about the centre of a 64^2 grid): along the
    # centre row the tumour occupies the cells whose centres lie within the disk
    wl = workloads.make(0)
    lo, hi = oracle.front(wl.V[0], 0, 32, 0.5)
    assert (lo, hi) == (26, 37) and oracle.front(wl.V[0], 1, 32, 0.5) == (26, 37)


# ---------------------------------------------------------------------------------------------
# Non-uniform step size dt_k (NEXT-2; the RULE is reading A6 and "parity unpinned": PAPER.md:62
# prints no formula.  What is pinned here is its arithmetic and the time loop around it.)
# ---------------------------------------------------------------------------------------------
def test_adaptive_dt_worked_values_and_brute_force():
    # worked value: A = diag(0.02, 0.01), b = 0 => lambda_max = 0.02; U = 0.75 everywhere and
    # alpha = 0.2 => alpha (1 - U) = 0.05 > lambda_max; h = 0.5, safety = 0.1 => 0.1 * 0.25 / 0.05
    a, b, c = np.full((3, 4), 0.02), np.zeros((3, 4)), np.full((3, 4), 0.01)
    U = np.full((3, 4), 0.75)
    assert oracle.adaptive_dt(U, a, b, c, 0.2, 0.5, safety=0.1) == pytest.approx(0.5, rel=1e-15)
    # alpha (1 - U) below lambda_max: the tensor decides, 0.1 * 0.25 / 0.02
    assert oracle.adaptive_dt(U, a, b, c, 0.04, 0.5, safety=0.1) == pytest.approx(1.25, rel=1e-15)
    # dx != dy: the smaller mesh size enters squared
    assert oracle.adaptive_dt(U, a, b, c, 0.2, 0.5, dy=0.25, safety=0.1) == pytest.approx(0.125, rel=1e-15)
    # brute force on a random batch: max over simulations and cells written as loops
    rng = np.random.default_rng(77)
    Ub = rng.uniform(-0.1, 1.1, (3, 5, 6))      # includes U > 1 (1 - U < 0) and U < 0
    al = np.array([0.03, 0.5, 0.2])
    aa, bb, cc = rng.uniform(5e-3, 2e-2, (5, 6)), rng.uniform(-4e-3, 4e-3, (5, 6)), rng.uniform(5e-3, 2e-2, (5, 6))
    rate = max(np.linalg.eigvalsh(np.array([[aa[j, i], bb[j, i]], [bb[j, i], cc[j, i]]]))[1]
               for j in range(5) for i in range(6))
    for s in range(3):
        for j in range(5):
            for i in range(6):
                rate = max(rate, al[s] * (1.0 - Ub[s, j, i]))
    assert oracle.adaptive_dt(Ub, aa, bb, cc, al, 0.25, safety=0.2) == pytest.approx(0.2 * 0.0625 / rate, rel=1e-14)
    # where the V diffusivity sits at its bound alpha (some cell has U = 0) the rule IS reading
    # A6's max_stable_dt
    Ub[1, 2, 3] = 0.0
    Ub = np.clip(Ub, 0.0, 1.0)
    assert oracle.adaptive_dt(Ub, aa, bb, cc, al, 0.25, safety=0.2) == \
        oracle.max_stable_dt(aa, bb, cc, al, 0.25, safety=0.2)


def test_step_adaptive_is_the_step_with_hand_fed_step_sizes():
    w = workloads.random_problem(61, 20, 14, batch=2)
    al = np.array([0.2, 0.3])                        # alpha (1 - U) above lambda_max ~ 0.035: U drives dt_k
    U0 = 0.6 + 0.4 * w.U                              # 1 - U starts in [0, 0.4] and grows as W kills U
    kw = dict(r=w.r, d=w.d * 4.0, alpha=al, c_r=w.c_r)
    U, V, W, t, dts = oracle.step_adaptive(U0, w.V, w.W, w.a, w.b, w.c, n=23, safety=0.2, every_k=5,
                                           dx=w.h, **kw)
    assert len(dts) == 5 and t == pytest.approx(sum(dts[:4]) * 5 + dts[4] * 3, rel=1e-15)
    assert dts[0] > dts[-1] > 0                       # U decays => the V diffusivity bound grows
    # replay by hand: the same groups through `step`, dt_k recomputed from the definition
    Uh, Vh, Wh = U0.copy(), w.V.copy(), w.W.copy()
    for g, n in enumerate((5, 5, 5, 5, 3)):
        rate = max(oracle.lambda_max(w.a, w.b, w.c), max(al[s] * (1.0 - Uh[s]).max() for s in range(2)))
        dt = 0.2 * w.h ** 2 / rate
        assert dt == pytest.approx(dts[g], rel=1e-15)
        for s in range(2):
            Uh[s], Vh[s], Wh[s] = oracle.step(Uh[s], Vh[s], Wh[s], w.a, w.b, w.c, r=w.r[s], d=4.0 * w.d[s],
                                              alpha=al[s], c_r=w.c_r[s], n=n, dt=dts[g], dx=w.h)
    assert np.array_equal(U, Uh) and np.array_equal(V, Vh) and np.array_equal(W, Wh)
    # alpha far below lambda_max: dt_k is constant and the run IS the fixed-step run, bit for bit
    U2, V2, W2, t2, dts2 = oracle.step_adaptive(w.U[0], w.V[0], w.W[0], w.a, w.b, w.c, r=1.0, d=3.0,
                                                alpha=1e-4, c_r=1.0, n=9, safety=0.2, every_k=2, dx=w.h)
    dt = oracle.max_stable_dt(w.a, w.b, w.c, 1e-4, w.h, safety=0.2)
    assert dts2 == [dt] * 5
    ref = oracle.step(w.U[0], w.V[0], w.W[0], w.a, w.b, w.c, r=1.0, d=3.0, alpha=1e-4, c_r=1.0, n=9,
                      dt=dt, dx=w.h)
    assert all(np.array_equal(x, y) for x, y in zip((U2, V2, W2), ref))
