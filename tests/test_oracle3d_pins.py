"""Pins of the 3-D oracle (oracle/gg3_oracle.cpp) against what the mathematics and the pinned 2-D
oracle fix.  CPU only (-m "not gpu").  None of these re-types the oracle's weight table: the brute
force below evaluates NESTED CENTRAL DIFFERENCES on the mirror-extended arrays (a different formula
route), the closed forms come from calculus, the reductions from the 2-D oracle, which is pinned to
the paper's printed tables (tests/test_oracle_pins.py).

Scheme = DESIGN.md reading A13 (the paper names 3-D as future work only): eq. (3) and
Tables 1-2 one dimension up."""
import itertools

import numpy as np
import pytest

import oracle


def rng(seed):
    return np.random.default_rng([200601748, 3, seed])


def spd_tensor(g, shape, off=0.3):
    """six fields (axx, ayy, azz, axy, axz, ayz), positive definite in every cell"""
    d = [1e-2 * (0.5 + g.random(shape)) for _ in range(3)]
    beta = [off * (2.0 * g.random(shape) - 1.0) for _ in range(3)]
    xy = beta[0] * np.sqrt(d[0] * d[1])
    xz = beta[1] * np.sqrt(d[0] * d[2])
    yz = beta[2] * np.sqrt(d[1] * d[2])
    return d[0], d[1], d[2], xy, xz, yz


# ---------------------------------------------------------------------------------------------
# brute force: nested central differences on mirror-extended arrays (pure Python loops)
# ---------------------------------------------------------------------------------------------
def mirror(P, sx=1, sy=1, sz=1):
    """one-cell ghost frame: even (+1) or odd (-1) mirror per axis (reading A2 in 3-D)"""
    nz, ny, nx = P.shape
    Q = np.zeros((nz + 2, ny + 2, nx + 2))
    for k in range(-1, nz + 1):
        for j in range(-1, ny + 1):
            for i in range(-1, nx + 1):
                f = 1.0
                kk, jj, ii = k, j, i
                if k < 0 or k >= nz:
                    kk, f = (0 if k < 0 else nz - 1), f * sz
                if j < 0 or j >= ny:
                    jj, f = (0 if j < 0 else ny - 1), f * sy
                if i < 0 or i >= nx:
                    ii, f = (0 if i < 0 else nx - 1), f * sx
                Q[k + 1, j + 1, i + 1] = f * P[kk, jj, ii]
    return Q


def brute_D2(tensor, W, h):
    """div(A grad W) by nested differences: the diagonal part as a difference of face fluxes with
    arithmetic face means, every mixed part d_p(a_pq d_q W) as a central difference (over 2 h_p) of
    cell-centred central differences (over 2 h_q)"""
    axx, ayy, azz, axy, axz, ayz = tensor
    nz, ny, nx = W.shape
    Wm = mirror(W)
    diag = [mirror(axx), mirror(ayy), mirror(azz)]
    offd = {(0, 1): mirror(axy, -1, -1, 1), (0, 2): mirror(axz, -1, 1, -1), (1, 2): mirror(ayz, 1, -1, -1)}
    e = [np.array(v) for v in ((0, 0, 1), (0, 1, 0), (1, 0, 0))]   # unit steps along x, y, z in (k, j, i) order
    out = np.zeros_like(W)
    for k, j, i in itertools.product(range(nz), range(ny), range(nx)):
        c = np.array((k + 1, j + 1, i + 1))
        at = lambda A, p: A[tuple(p)]
        s = 0.0
        for p in range(3):
            fp = 0.5 * (at(diag[p], c) + at(diag[p], c + e[p])) * (at(Wm, c + e[p]) - at(Wm, c)) / h[p]
            fm = 0.5 * (at(diag[p], c - e[p]) + at(diag[p], c)) * (at(Wm, c) - at(Wm, c - e[p])) / h[p]
            s += (fp - fm) / h[p]
        for (p, q), A in offd.items():
            for a_, b_ in ((p, q), (q, p)):     # d_a (a_pq d_b W)
                def inner(cc):   # a_pq d_b W at a cell (ghost cells of W: one more mirror step)
                    return at(A, cc) * (wat(cc + e[b_]) - wat(cc - e[b_])) / (2.0 * h[b_])
                def wat(cc):     # W with double ghosts resolved by mirroring indices
                    kk, jj, ii = (int(min(max(v, 1), n)) for v, n in zip(cc, (nz, ny, nx)))
                    return Wm[kk, jj, ii]
                s += (inner(c + e[a_]) - inner(c - e[a_])) / (2.0 * h[a_])
        out[k, j, i] = s
    return out


def brute_D1(U, V, h):
    nz, ny, nx = U.shape
    Um, Vm = mirror(U), mirror(V)
    e = [np.array(v) for v in ((0, 0, 1), (0, 1, 0), (1, 0, 0))]
    out = np.zeros_like(U)
    for k, j, i in itertools.product(range(nz), range(ny), range(nx)):
        c = np.array((k + 1, j + 1, i + 1))
        s = 0.0
        for p in range(3):
            fp = (1.0 - 0.5 * (Um[tuple(c)] + Um[tuple(c + e[p])])) * (Vm[tuple(c + e[p])] - Vm[tuple(c)]) / h[p]
            fm = (1.0 - 0.5 * (Um[tuple(c - e[p])] + Um[tuple(c)])) * (Vm[tuple(c)] - Vm[tuple(c - e[p])]) / h[p]
            s += (fp - fm) / h[p]
        out[k, j, i] = s
    return out


@pytest.mark.parametrize("shape,h", [((3, 3, 3), (1.0, 1.0, 1.0)), ((4, 3, 5), (0.5, 0.25, 0.125)), ((2, 2, 2), (1.0, 2.0, 0.5))])
def test_D2_matches_nested_central_differences(shape, h):
    g = rng(1)
    T = spd_tensor(g, shape)
    W = g.random(shape)
    got = oracle.D2_3d(T, W, *h)
    want = brute_D2(T, W, h)
    scale = np.max(np.abs(want)) + 1e-300
    assert np.max(np.abs(got - want)) <= 1e-13 * scale


@pytest.mark.parametrize("shape,h", [((3, 4, 3), (1.0, 1.0, 1.0)), ((2, 3, 4), (0.5, 0.25, 2.0))])
def test_D1_matches_flux_differences(shape, h):
    g = rng(2)
    U, V = g.random(shape), g.random(shape)
    got = oracle.D1_3d(U, V, *h)
    want = brute_D1(U, V, h)
    assert np.max(np.abs(got - want)) <= 1e-13 * (np.max(np.abs(want)) + 1e-300)


# ---------------------------------------------------------------------------------------------
# closed forms (interior cells: central differences are exact on these polynomials)
# ---------------------------------------------------------------------------------------------
def grid(shape, h):
    nz, ny, nx = shape
    z, y, x = np.meshgrid((np.arange(nz) + 0.5) * h[2], (np.arange(ny) + 0.5) * h[1], (np.arange(nx) + 0.5) * h[0], indexing="ij")
    return x, y, z


def const_tensor(shape, vals):
    return tuple(np.full(shape, v) for v in vals)


@pytest.mark.parametrize("W_of,entry,value", [
    (lambda x, y, z: x * x, 0, 2.0), (lambda x, y, z: y * y, 1, 2.0), (lambda x, y, z: z * z, 2, 2.0),
    (lambda x, y, z: x * y, 3, 2.0), (lambda x, y, z: x * z, 4, 2.0), (lambda x, y, z: y * z, 5, 2.0),
    (lambda x, y, z: x * y, 4, 0.0), (lambda x, y, z: x * z, 5, 0.0), (lambda x, y, z: y * z, 3, 0.0),
    (lambda x, y, z: x * x, 3, 0.0), (lambda x, y, z: z * z, 0, 0.0)])
def test_D2_polynomials_per_tensor_entry(W_of, entry, value):
    """div(A grad W) with ONE constant non-zero tensor entry a: W = p^2 -> 2 a_pp; W = p q -> 2 a_pq;
    anything else -> 0.  A wrong sign, factor or plane of a cross term fails one of these."""
    shape, h = (6, 5, 7), (0.5, 0.25, 0.2)
    x, y, z = grid(shape, h)
    vals = [0.0] * 6
    vals[entry] = 0.7
    got = oracle.D2_3d(const_tensor(shape, vals), W_of(x, y, z), *h)
    inner = got[1:-1, 1:-1, 1:-1]
    assert np.max(np.abs(inner - value * 0.7)) <= 1e-12


def test_D2_plane_wave_symbol():
    """constant A, W = cos(k.x): interior value = -[sum_p a_pp (2 - 2 cos(k_p h_p))/h_p^2
    + 2 sum_{p<q} a_pq sin(k_p h_p) sin(k_q h_q)/(h_p h_q)] W  (the discrete symbol)"""
    shape, h = (8, 9, 10), (0.3, 0.2, 0.25)
    kv = (1.3, -0.7, 2.1)
    x, y, z = grid(shape, h)
    W = np.cos(kv[0] * x + kv[1] * y + kv[2] * z)
    vals = (1.1, 0.9, 1.3, 0.35, -0.25, 0.15)
    got = oracle.D2_3d(const_tensor(shape, vals), W, *h)
    s = [np.sin(kv[p] * h[p]) / h[p] for p in range(3)]
    dd = [(2.0 - 2.0 * np.cos(kv[p] * h[p])) / h[p] ** 2 for p in range(3)]
    sym = -(vals[0] * dd[0] + vals[1] * dd[1] + vals[2] * dd[2] +
            2.0 * (vals[3] * s[0] * s[1] + vals[4] * s[0] * s[2] + vals[5] * s[1] * s[2]))
    inner = (slice(1, -1),) * 3
    assert np.max(np.abs(got[inner] - sym * W[inner])) <= 1e-11


# ---------------------------------------------------------------------------------------------
# reductions to the pinned 2-D oracle, axis permutations
# ---------------------------------------------------------------------------------------------
def test_z_uniform_data_is_the_2d_oracle_bit_for_bit():
    g = rng(5)
    ny, nx, nz = 7, 9, 4
    a, c = 1e-2 * (0.5 + g.random((ny, nx))), 1e-2 * (0.5 + g.random((ny, nx)))
    b = 0.6 * (2 * g.random((ny, nx)) - 1) * np.sqrt(a * c)
    U, V, W = g.random((ny, nx)), g.random((ny, nx)), g.random((ny, nx))
    par = dict(r=1.0, d=3.0, alpha=1e-3, c_r=0.7)
    rep = lambda P: np.repeat(P[None], nz, axis=0)
    zero = np.zeros((nz, ny, nx))
    T = (rep(a), rep(c), rep(1e-2 * (0.5 + g.random((ny, nx)))), rep(b), zero, zero)
    dt, dx, dy = 2e-3, 0.5, 0.25
    ref = oracle.step(U, V, W, a, b, c, n=5, dt=dt, dx=dx, dy=dy, **par)
    got = oracle.step3d(rep(U), rep(V), rep(W), T, n=5, dt=dt, dx=dx, dy=dy, dz=0.3, **par)
    for g3, r2 in zip(got, ref):
        for k in range(nz):
            assert np.array_equal(g3[k], r2)


PERMS = {  # new axes (x', y', z') = old axes in this order; tensor entries follow
    (1, 2, 0): None, (2, 0, 1): None, (1, 0, 2): None, (0, 2, 1): None, (2, 1, 0): None}


def permute(fields, tensor, h, perm):
    """relabel the coordinate axes: new axis p is old axis perm[p] (arrays are [z][y][x])"""
    # array axis of coordinate axis p (x=0,y=1,z=2) is 2-p
    axes = tuple(2 - perm[2 - ax] for ax in range(3))
    tr = lambda P: np.ascontiguousarray(np.transpose(P, axes))
    diag = [tensor[0], tensor[1], tensor[2]]
    off = {frozenset((0, 1)): tensor[3], frozenset((0, 2)): tensor[4], frozenset((1, 2)): tensor[5]}
    nd = [tr(diag[perm[p]]) for p in range(3)]
    no = [tr(off[frozenset((perm[p], perm[q]))]) for p, q in ((0, 1), (0, 2), (1, 2))]
    return [tr(F) for F in fields], tuple(nd + no), tuple(h[perm[p]] for p in range(3)), axes


@pytest.mark.parametrize("perm", list(PERMS))
def test_axis_permutations(perm):
    g = rng(6)
    shape, h = (4, 5, 6), (0.5, 0.4, 0.3)
    T = spd_tensor(g, shape)
    F = [g.random(shape) for _ in range(3)]
    par = dict(r=0.8, d=2.5, alpha=2e-3, c_r=1.1, n=4, dt=1e-3)
    ref = oracle.step3d(*F, T, dx=h[0], dy=h[1], dz=h[2], **par)
    F2, T2, h2, axes = permute(F, T, h, perm)
    got = oracle.step3d(*F2, T2, dx=h2[0], dy=h2[1], dz=h2[2], **par)
    for gf, rf in zip(got, ref):
        assert np.max(np.abs(gf - np.transpose(rf, axes))) <= 1e-14
    # non-vacuity: the permuted problem is a different array problem
    assert not np.allclose(got[2], ref[2].reshape(got[2].shape)) or shape[0] == shape[1] == shape[2]


@pytest.mark.parametrize("axis", [1, 2])
def test_uniform_along_y_or_x_reduces_to_2d(axis):
    """data uniform along y (array axis 1) or x (array axis 2) with the off-diagonals that involve
    that axis set to zero = the 2-D oracle on the remaining two axes"""
    g = rng(7)
    n1, n2, nu = 6, 5, 3
    a, c = 1e-2 * (0.5 + g.random((n1, n2))), 1e-2 * (0.5 + g.random((n1, n2)))
    b = 0.5 * (2 * g.random((n1, n2)) - 1) * np.sqrt(a * c)
    U, V, W = (g.random((n1, n2)) for _ in range(3))
    par = dict(r=1.0, d=2.0, alpha=1e-3, c_r=0.5, n=6, dt=2e-3)
    ref = oracle.step(U, V, W, a, b, c, dx=0.4, dy=0.3, **par)   # 2-D: x = fast axis (n2), y = slow axis (n1)
    ins = lambda P: np.ascontiguousarray(np.repeat(np.expand_dims(P, axis), nu, axis=axis))
    other = ins(1e-2 * (0.5 + g.random((n1, n2))))
    zero = np.zeros_like(other)
    if axis == 1:    # arrays [z][y][x] = [n1][uniform][n2]: 2-D (x, y) -> 3-D (x, z)
        T = (ins(a), other, ins(c), zero, ins(b), zero)
        got = oracle.step3d(ins(U), ins(V), ins(W), T, dx=0.4, dy=0.7, dz=0.3, **par)
    else:            # arrays [n1][n2][uniform]: 2-D (x, y) -> 3-D (y, z)
        T = (other, ins(a), ins(c), zero, zero, ins(b))
        got = oracle.step3d(ins(U), ins(V), ins(W), T, dx=0.7, dy=0.4, dz=0.3, **par)
    for g3, r2 in zip(got, ref):
        for u in range(nu):
            assert np.max(np.abs(np.take(g3, u, axis=axis) - r2)) <= 1e-15


# ---------------------------------------------------------------------------------------------
# conservation, scalar recursion, equilibria
# ---------------------------------------------------------------------------------------------
def test_mass_conservation_with_all_cross_terms():
    """reactions off: sum W (any positive-definite heterogeneous tensor, all three off-diagonals
    non-zero) and sum V are conserved under the mirrored (zero-flux) boundaries"""
    g = rng(8)
    shape = (5, 6, 7)
    T = spd_tensor(g, shape)
    U, V, W = g.random(shape), g.random(shape), g.random(shape)
    got = oracle.step3d(U, V, W, T, r=0.0, d=0.0, alpha=5e-3, c_r=0.0, n=20, dt=2e-2, dx=0.5, dy=0.4, dz=0.6)
    assert abs(got[2].sum() - W.sum()) <= 1e-12 * W.sum()
    assert abs(got[1].sum() - V.sum()) <= 1e-12 * V.sum()
    # an even mirror of an off-diagonal entry (the rejected reading) would leak: non-vacuity
    leak = oracle.D2_3d(T, W, 0.5, 0.4, 0.6).sum()
    assert abs(leak) <= 1e-12 * np.abs(oracle.D2_3d(T, W, 0.5, 0.4, 0.6)).sum()


def test_uniform_data_is_the_scalar_recursion():
    shape = (3, 4, 5)
    g = rng(9)
    T = spd_tensor(g, shape)
    u, v, w = 0.3, 0.6, 0.2
    r, d, c_r, dt = 0.9, 4.0, 1.2, 1e-2
    got = oracle.step3d(np.full(shape, u), np.full(shape, v), np.full(shape, w), T, r=r, d=d, alpha=1e-3, c_r=c_r, n=7, dt=dt, dx=1.0)
    for _ in range(7):
        u, v, w = u + dt * u * (1.0 - u) - d * dt * u * w, v + r * dt * v * (1.0 - v), w + c_r * dt * (v - w)
    assert np.all(got[0] == u) and np.all(got[1] == v) and np.all(got[2] == w)


@pytest.mark.parametrize("state", [(1.0, 0.0, 0.0), (0.0, 1.0, 1.0), (0.0, 0.0, 0.0)])
def test_equilibria_are_stationary(state):
    shape = (4, 4, 4)
    T = spd_tensor(rng(10), shape)
    F = [np.full(shape, s) for s in state]
    got = oracle.step3d(*F, T, r=1.0, d=10.0, alpha=1e-3, c_r=1.0, n=10, dt=1e-2, dx=0.25)
    for gq, f in zip(got, F):
        assert np.array_equal(gq, f)


def test_thread_count_independence():
    g = rng(11)
    shape = (6, 5, 7)
    T = spd_tensor(g, shape)
    F = [g.random(shape) for _ in range(3)]
    par = dict(r=1.0, d=3.0, alpha=1e-3, c_r=1.0, n=3, dt=1e-3, dx=0.5)
    a = oracle.step3d(*F, T, threads=1, **par)
    b = oracle.step3d(*F, T, threads=4, **par)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
