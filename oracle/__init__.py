"""CPU oracle for the Gatenby-Gawlinski finite-volume step -- TEST INFRASTRUCTURE, not product.

Thin ctypes front for oracle/gg_oracle.cpp (plain fp64 C++, literal Table-1 / Table-2 stencils,
eq. (3) of arXiv 2006.01748; see that file's header for citations and the pins that hold it).

Only tests/, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` / `--impl reference` legs may
import this package.  It imports nothing from paper_2006_01748_b200 and is imported by nothing
there.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import build as _build

_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        lib.gg_oracle_D1.restype = ctypes.c_int
        lib.gg_oracle_D1.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                     _dp, _dp, _dp]
        lib.gg_oracle_D2.restype = ctypes.c_int
        lib.gg_oracle_D2.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                     _dp, _dp, _dp, _dp, _dp]
        lib.gg_oracle_step.restype = ctypes.c_int
        lib.gg_oracle_step.argtypes = ([ctypes.c_int, ctypes.c_int] + [ctypes.c_double] * 6 +
                                       [_dp] * 6 + [ctypes.c_longlong, ctypes.c_double,
                                                    ctypes.c_int])
        lib.gg_oracle_max_threads.restype = ctypes.c_int
        lib.gg_oracle_max_threads.argtypes = []
        # the 3-D extension (oracle/gg3_oracle.cpp)
        lib.gg3_oracle_D1.restype = ctypes.c_int
        lib.gg3_oracle_D1.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [_dp] * 3
        lib.gg3_oracle_D2.restype = ctypes.c_int
        lib.gg3_oracle_D2.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 3 + [_dp] * 8
        lib.gg3_oracle_step.restype = ctypes.c_int
        lib.gg3_oracle_step.argtypes = ([ctypes.c_int] * 3 + [ctypes.c_double] * 7 + [_dp] * 9 +
                                        [ctypes.c_longlong, ctypes.c_double, ctypes.c_int])
        _lib = lib
    return _lib


def _c(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(x: np.ndarray):
    return x.ctypes.data_as(_dp)


def max_threads() -> int:
    return int(load().gg_oracle_max_threads())


def D1(U, V, dx: float, dy: float) -> np.ndarray:
    """D1(V;U), Table 1, mirrored ghosts.  U, V: [ny][nx]."""
    U, V = _c(U), _c(V)
    ny, nx = U.shape
    out = np.empty_like(U)
    rc = load().gg_oracle_D1(nx, ny, dx, dy, _p(U), _p(V), _p(out))
    if rc != 0:
        raise ValueError("gg_oracle_D1: bad argument")
    return out


def D2(a, b, c, W, dx: float, dy: float) -> np.ndarray:
    """D2(W;A), Table 2, mirrored ghosts with b odd.  All [ny][nx]."""
    a, b, c, W = _c(a), _c(b), _c(c), _c(W)
    ny, nx = W.shape
    out = np.empty_like(W)
    rc = load().gg_oracle_D2(nx, ny, dx, dy, _p(a), _p(b), _p(c), _p(W), _p(out))
    if rc != 0:
        raise ValueError("gg_oracle_D2: bad argument")
    return out


def step(U, V, W, a, b, c, *, r: float, d: float, alpha: float, c_r: float, n: int, dt: float,
         dx: float, dy: float | None = None, threads: int = 0):
    """n explicit Euler steps of eq. (3).  Returns new (U, V, W); inputs untouched.

    `c` is the tensor entry c_T(x,y) of eq. (2); `c_r` the reaction parameter eq. (1) calls c.
    threads <= 0: all cores OpenMP sees (results are bit-identical for any thread count).
    """
    if dy is None:
        dy = dx
    U, V, W = _c(U).copy(), _c(V).copy(), _c(W).copy()
    a, b, c = _c(a), _c(b), _c(c)
    ny, nx = U.shape
    for x in (V, W, a, b, c):
        if x.shape != (ny, nx):
            raise ValueError("shape mismatch")
    rc = load().gg_oracle_step(nx, ny, dx, dy, r, d, alpha, c_r, _p(a), _p(b), _p(c), _p(U), _p(V),
                               _p(W), int(n), float(dt), int(threads))
    if rc != 0:
        raise ValueError("gg_oracle_step: bad argument")
    return U, V, W


# ---------------------------------------------------------------------------------------------
# Reductions next to the step.  Plain NumPy, written out.
# Pins: tests/test_oracle_pins.py (brute-force loops on tiny grids, eigvalsh, closed forms).
# "parity unpinned": the step-size RULE of max_stable_dt (reading A6; the paper prints none).
# ---------------------------------------------------------------------------------------------
DIAG_NAMES = ("sum_U", "sum_V", "sum_W", "gap_cells", "tumour_cells", "min_W", "max_U", "max_W",
              "nonfinite_cells")


def diagnostics(U, V, W, eps: float) -> np.ndarray:
    """Diagnostics of one state [ny][nx], in the order DIAG_NAMES: the sums of the three fields,
    the number of interstitial-gap cells (U < eps and V < eps: neither cell type present, the gap
    between the fronts of PAPER.md:100-111), the number of tumour cells (V >= 1/2), min W, max U,
    max W (NaNs skipped, as fmin / fmax do), and the number of cells where U, V or W is not finite.
    Everything in fp64."""
    U, V, W = _c(U), _c(V), _c(W)
    return np.array([
        np.sum(U), np.sum(V), np.sum(W),
        float(np.count_nonzero((U < eps) & (V < eps))),
        float(np.count_nonzero(V >= 0.5)),
        np.nanmin(W) if np.isfinite(W).any() or np.isinf(W).any() else np.inf,
        np.nanmax(U) if not np.isnan(U).all() else -np.inf,
        np.nanmax(W) if not np.isnan(W).all() else -np.inf,
        float(np.count_nonzero(~(np.isfinite(U) & np.isfinite(V) & np.isfinite(W))))], dtype=np.float64)


def lambda_max(a, b, c) -> float:
    """max over cells of the larger eigenvalue of the tensor [[a,b],[b,c]] of eq. (2)
    (PAPER.md:40): (a+c)/2 + sqrt(((a-c)/2)^2 + b^2)."""
    a, b, c = _c(a), _c(b), _c(c)
    return float(np.max(0.5 * (a + c) + np.sqrt((0.5 * (a - c)) ** 2 + b ** 2)))


def max_stable_dt(a, b, c, alpha, dx: float, dy: float | None = None, safety: float = 0.2) -> float:
    """DESIGN.md reading A6 (the paper prints no formula):
    safety * min(dx,dy)^2 / max(max alpha, lambda_max(A)).

    PARITY UNPINNED as far as the RULE goes: the paper says only that the host recomputes the step
    "to ensure numerical stability"; nothing it prints fixes this formula (lambda_max itself is
    pinned against LAPACK and closed forms, and the arithmetic of the rule against worked values)."""
    if dy is None:
        dy = dx
    rate = max(float(np.max(alpha)), lambda_max(a, b, c))
    return safety * min(dx, dy) ** 2 / rate


def front(F, axis: int, index: int, level: float):
    """First and last cell index along row `index` (axis 0: the line runs along x) or column
    `index` (axis 1) of one field [ny][nx] where the field is >= level; (-1, -1) if none.  The
    positions of the tumour and acid fronts along a ray."""
    F = _c(F)
    line = F[index, :] if axis == 0 else F[:, index]
    idx = np.nonzero(line >= level)[0]
    return (int(idx[0]), int(idx[-1])) if idx.size else (-1, -1)


# ---------------------------------------------------------------------------------------------
# Non-uniform step size dt_k ("nonuniform step-size dt_k ...
# computed after each iteration", PAPER.md:127-128 steps 3-4).  Plain NumPy + the C step above.
#
# PARITY UNPINNED as far as the RULE goes (reading A6: the paper prints no formula).
# What IS pinned (tests/test_oracle_pins.py): the rule's arithmetic against worked values and
# brute-force loops, its reduction to max_stable_dt when the V diffusivity alpha (1 - U) is at its
# bound alpha, the time loop against `step` with hand-fed step sizes, the clock against sum dt_k.
# ---------------------------------------------------------------------------------------------
def adaptive_dt(U, a, b, c, alpha, dx: float, dy: float | None = None, safety: float = 0.2) -> float:
    """dt_k = safety * min(dx,dy)^2 / max(lambda_max(A), max_s alpha_s * max_ij (1 - U_s,ij)).

    U: [ny][nx] or [batch][ny][nx]; alpha: scalar or [batch].  lambda_max(A) bounds the W
    diffusion, alpha (1 - U) is the diffusivity of the V equation (eq. (1)) at the
    current time level; one step size for the whole batch."""
    if dy is None:
        dy = dx
    U = _c(U)
    if U.ndim == 2:
        U = U[None]
    al = np.broadcast_to(np.asarray(alpha, dtype=np.float64), (U.shape[0],))
    rate = lambda_max(a, b, c)
    for s in range(U.shape[0]):
        rate = max(rate, float(al[s] * np.max(1.0 - U[s])))
    hmin = min(dx, dy)
    return safety * hmin * hmin / rate


def step_adaptive(U, V, W, a, b, c, *, r, d, alpha, c_r, n: int, safety: float, every_k: int,
                  dx: float, dy: float | None = None, threads: int = 0):
    """n explicit steps of eq. (3) with dt_k re-evaluated by `adaptive_dt` from the current U
    before every group of `every_k` steps (the last group may be shorter).  U, V, W:
    [batch][ny][nx] (or [ny][nx] for one simulation); r, d, alpha, c_r scalars or [batch].
    Returns (U, V, W, time, dts) with time = sum of all step sizes and dts = the dt_k of every
    group."""
    if dy is None:
        dy = dx
    single = np.ndim(U) == 2
    U, V, W = (np.array(x, dtype=np.float64, ndmin=3) for x in (U, V, W))
    B = U.shape[0]
    par = [np.broadcast_to(np.asarray(p, dtype=np.float64), (B,)) for p in (r, d, alpha, c_r)]
    t, left, dts = 0.0, int(n), []
    while left > 0:
        g = min(left, int(every_k))
        dt = adaptive_dt(U, a, b, c, par[2], dx, dy, safety)
        for s in range(B):
            U[s], V[s], W[s] = step(U[s], V[s], W[s], a, b, c, r=par[0][s], d=par[1][s],
                                    alpha=par[2][s], c_r=par[3][s], n=g, dt=dt, dx=dx, dy=dy,
                                    threads=threads)
        t += dt * g
        dts.append(dt)
        left -= g
    if single:
        U, V, W = U[0], V[0], W[0]
    return U, V, W, t, dts


# ---------------------------------------------------------------------------------------------
# Three-dimensional extension.  Front for oracle/gg3_oracle.cpp:
# the construction of eq. (3) and Tables 1-2 one dimension up (reading A13; the paper
# prints no 3-D scheme).  Arrays are [nz][ny][nx]; the tensor is the six arrays
# (axx, ayy, azz, axy, axz, ayz).  Pins: tests/test_oracle3d_pins.py.
# ---------------------------------------------------------------------------------------------
def D1_3d(U, V, dx: float, dy: float, dz: float) -> np.ndarray:
    """Seven-point D1(V;U) (Table 1 with the two z entries added), mirrored ghosts."""
    U, V = _c(U), _c(V)
    nz, ny, nx = U.shape
    out = np.empty_like(U)
    if load().gg3_oracle_D1(nx, ny, nz, dx, dy, dz, _p(U), _p(V), _p(out)) != 0:
        raise ValueError("gg3_oracle_D1: bad argument")
    return out


def D2_3d(tensor, W, dx: float, dy: float, dz: float) -> np.ndarray:
    """Nineteen-point D2(W;A): Table 2's face and corner entries in each coordinate plane."""
    T = [_c(t) for t in tensor]
    W = _c(W)
    nz, ny, nx = W.shape
    out = np.empty_like(W)
    if load().gg3_oracle_D2(nx, ny, nz, dx, dy, dz, *[_p(t) for t in T], _p(W), _p(out)) != 0:
        raise ValueError("gg3_oracle_D2: bad argument")
    return out


def step3d(U, V, W, tensor, *, r: float, d: float, alpha: float, c_r: float, n: int, dt: float,
           dx: float, dy: float | None = None, dz: float | None = None, threads: int = 0):
    """n explicit Euler steps of eq. (3) in three dimensions.  Returns new (U, V, W)."""
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    U, V, W = _c(U).copy(), _c(V).copy(), _c(W).copy()
    T = [_c(t) for t in tensor]
    nz, ny, nx = U.shape
    for x in (V, W, *T):
        if x.shape != (nz, ny, nx):
            raise ValueError("shape mismatch")
    rc = load().gg3_oracle_step(nx, ny, nz, dx, dy, dz, r, d, alpha, c_r, *[_p(t) for t in T],
                                _p(U), _p(V), _p(W), int(n), float(dt), int(threads))
    if rc != 0:
        raise ValueError("gg3_oracle_step: bad argument")
    return U, V, W
