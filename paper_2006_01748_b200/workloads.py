"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module holds NONE of the method's arithmetic: it only builds parameter values, tensor
coefficient fields, initial states and the step size handed to `gg_step`.  It is the one module
both the CUDA path's tests/bench and the CPU oracle's tests read, so that both sides see the same
arrays.  NumPy only; no torch, no CUDA, no oracle import.

The paper's own inputs (tensor fields "derived from the experimental setting"; the
Fig. 2 parameters) are not published, so every workload here is synthetic and
stands in for them: a square Petri dish of healthy tissue U=1 with tumour seeds V=1,
no acid, an anisotropic / heterogeneous positive-definite tensor, d on both
sides of 1.  The recipe for each config is spelled out in DESIGN.md §5.

Conventions (readings A1, A6, A11):
  * nx x ny cells tile [0,L]^2 with L = nx*h; cell (i,j) has centre ((i+1/2)h, (j+1/2)h);
    arrays are [ny][nx], x fastest.
  * a disk contains a cell iff the cell centre lies within radius R of the disk centre.
  * state = indicator values, then += uniform[0,1e-3) noise on U, then on V (two full-array
    draws, U first), clipped to [0,1]; W = 0.
  * dt = 0.2*h^2 / max(alpha, lambda_max(A)), lambda_max = max over cells of the larger
    eigenvalue of [[a,b],[b,c]], evaluated once here in fp64.
  * one generator per config: np.random.default_rng([200601748, cfg]), draws in the order listed.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED = 200601748
H = 1.0 / 64.0


@dataclass
class Workload:
    name: str
    cfg: int
    nx: int
    ny: int
    h: float
    batch: int
    r: np.ndarray        # [batch]
    d: np.ndarray        # [batch]
    alpha: np.ndarray    # [batch]
    c_r: np.ndarray      # [batch]  (the reaction parameter eq. (1) calls c)
    a: np.ndarray        # [ny][nx] tensor entry a(x,y)
    b: np.ndarray        # [ny][nx] tensor entry b(x,y)
    c: np.ndarray        # [ny][nx] tensor entry c(x,y)  (c_T)
    U: np.ndarray        # [batch][ny][nx]
    V: np.ndarray
    W: np.ndarray
    dt: float
    steps: int
    dtypes: tuple = ("f64",)
    notes: dict = field(default_factory=dict)
    hy: float | None = None   # dy when the mesh is not square; None: dy = dx = h

    @property
    def dy(self) -> float:
        return self.h if self.hy is None else self.hy

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.batch

    @property
    def cell_updates(self) -> int:
        return self.cells * self.steps


def cell_centres(nx: int, ny: int, h: float):
    x = (np.arange(nx, dtype=np.float64) + 0.5) * h
    y = (np.arange(ny, dtype=np.float64) + 0.5) * h
    return x[None, :], y[:, None]


def lambda_max(a: np.ndarray, b: np.ndarray, c: np.ndarray) -> float:
    """Largest eigenvalue of [[a,b],[b,c]] over all cells (used by the dt rule only)."""
    lam = 0.5 * (a + c) + np.sqrt(0.25 * (a - c) ** 2 + b ** 2)
    return float(lam.max())


def dt_rule(h: float, alpha_max: float, a, b, c) -> float:
    return 0.2 * h * h / max(float(alpha_max), lambda_max(a, b, c))


def disk_state(rng, nx, ny, h, disks, noise=True):
    """U=1,V=0 outside the union of disks, U=0,V=1 inside; W=0; + noise on U then V; clip."""
    x, y = cell_centres(nx, ny, h)
    inside = np.zeros((ny, nx), dtype=bool)
    for (x0, y0, R) in disks:
        inside |= (x - x0) ** 2 + (y - y0) ** 2 <= R * R
    U = np.where(inside, 0.0, 1.0)
    V = np.where(inside, 1.0, 0.0)
    if noise:
        U = U + rng.uniform(0.0, 1e-3, (ny, nx))
        V = V + rng.uniform(0.0, 1e-3, (ny, nx))
    U = np.clip(U, 0.0, 1.0)
    V = np.clip(V, 0.0, 1.0)
    W = np.zeros((ny, nx))
    return U, V, W


def fourier_field(rng, nx, ny, h, modes=8):
    """Sum of `modes` seeded plane waves, wavenumbers 1..4 over L, normalised into [-1,1]."""
    L = nx * h
    x, y = cell_centres(nx, ny, h)
    f = np.zeros((ny, nx))
    amp = 0.0
    for _ in range(modes):
        kx = int(rng.integers(1, 5)) * int(rng.choice([-1, 1]))
        ky = int(rng.integers(1, 5))
        phi = float(rng.uniform(0.0, 2.0 * np.pi))
        A = float(rng.uniform(0.5, 1.0))
        f += A * np.cos(2.0 * np.pi * (kx * x + ky * y) / L + phi)
        amp += A
    return f / amp


def smooth_tensor(rng, nx, ny, h):
    f1 = fourier_field(rng, nx, ny, h)
    f2 = fourier_field(rng, nx, ny, h)
    g = fourier_field(rng, nx, ny, h)
    a = 1e-2 * (1.0 + 0.5 * f1)
    c = 1e-2 * (1.0 + 0.5 * f2)
    b = 0.8 * g * np.sqrt(a * c)
    return a, b, c


def banded_tensor(rng, nx, ny, nbands=6):
    a = np.empty((ny, nx))
    b = np.empty((ny, nx))
    c = np.empty((ny, nx))
    for k in range(nbands):
        j0, j1 = (k * ny) // nbands, ((k + 1) * ny) // nbands
        ak = float(rng.uniform(5e-3, 2e-2))
        ck = float(rng.uniform(5e-3, 2e-2))
        beta = float(rng.uniform(-0.9, 0.9))
        a[j0:j1, :] = ak
        c[j0:j1, :] = ck
        b[j0:j1, :] = beta * np.sqrt(ak * ck)
    return a, b, c


def _scalars(batch, r, d, alpha, c_r):
    f = lambda v: np.broadcast_to(np.asarray(v, dtype=np.float64), (batch,)).copy()
    return f(r), f(d), f(alpha), f(c_r)


def make(cfg: int, *, nx: int | None = None, ny: int | None = None, steps: int | None = None,
         d: float | None = None, batch: int | None = None) -> Workload:
    """Build BASELINE.json config `cfg` (0..4).

    nx / ny / steps / batch override the config's size with the SAME recipe (used by parity tests
    that need a grid the oracle finishes in seconds); d overrides the aggressiveness parameter
    (config 2 is swept over d in {2, 10, 20} from the same inputs).
    """
    rng = np.random.default_rng([SEED, cfg])
    h = H
    if cfg == 0:
        nx = nx or 64
        ny = ny or nx
        L = nx * h
        a = np.full((ny, nx), 1e-2)
        c = np.full((ny, nx), 1e-2)
        b = np.zeros((ny, nx))
        U, V, W = disk_state(rng, nx, ny, h, [(0.5 * L, 0.5 * ny * h, 0.1 * L)])
        r_, d_, al_, cr_ = _scalars(1, 1.0, 10.0 if d is None else d, 1e-3, 1.0)
        st = 200 if steps is None else steps
        name = f"cfg0 isotropic {nx}x{ny}"
        B = 1
        U, V, W = U[None], V[None], W[None]
    elif cfg == 1:
        nx = nx or 512
        ny = ny or nx
        L = nx * h
        a = np.full((ny, nx), 1.5e-2)
        c = np.full((ny, nx), 5e-3)
        b = np.full((ny, nx), 4e-3)
        U, V, W = disk_state(rng, nx, ny, h, [(0.5 * L, 0.5 * ny * h, 0.1 * L)])
        r_, d_, al_, cr_ = _scalars(1, 1.0, 10.0 if d is None else d, 1e-3, 1.0)
        st = 2000 if steps is None else steps
        name = f"cfg1 constant anisotropic {nx}x{ny}"
        B = 1
        U, V, W = U[None], V[None], W[None]
    elif cfg == 2:
        nx = nx or 2048
        ny = ny or nx
        L = nx * h
        a, b, c = smooth_tensor(rng, nx, ny, h)
        U, V, W = disk_state(rng, nx, ny, h, [(0.35 * L, 0.60 * ny * h, 0.05 * L)])
        r_, d_, al_, cr_ = _scalars(1, 1.0, 10.0 if d is None else d, 1e-3, 1.0)
        st = 10000 if steps is None else steps
        name = f"cfg2 smooth heterogeneous {nx}x{ny} d={float(d_[0]):g}"
        B = 1
        U, V, W = U[None], V[None], W[None]
    elif cfg == 3:
        nx = nx or 8192
        ny = ny or nx
        L = nx * h
        a, b, c = banded_tensor(rng, nx, ny)
        centres = rng.uniform(0.1 * L, 0.9 * L, (3, 2))
        if ny != nx:
            centres[:, 1] *= ny / nx
        U, V, W = disk_state(rng, nx, ny, h, [(cx, cy, 0.02 * L) for cx, cy in centres])
        r_, d_, al_, cr_ = _scalars(1, 1.0, 10.0 if d is None else d, 1e-3, 1.0)
        st = 1000 if steps is None else steps
        name = f"cfg3 layered discontinuous {nx}x{ny}"
        B = 1
        U, V, W = U[None], V[None], W[None]
    elif cfg == 4:
        nx = nx or 1024
        ny = ny or nx
        B = 64 if batch is None else batch
        L = nx * h
        a, b, c = smooth_tensor(rng, nx, ny, h)
        x, y = cell_centres(nx, ny, h)
        inside = (x - 0.35 * L) ** 2 + (y - 0.60 * ny * h) ** 2 <= (0.05 * L) ** 2
        U = np.empty((B, ny, nx))
        V = np.empty((B, ny, nx))
        for s in range(B):
            U[s] = np.clip(np.where(inside, 0.0, 1.0) + rng.uniform(0.0, 1e-3, (ny, nx)), 0.0, 1.0)
            V[s] = np.clip(np.where(inside, 1.0, 0.0) + rng.uniform(0.0, 1e-3, (ny, nx)), 0.0, 1.0)
        W = np.zeros((B, ny, nx))
        # sim s = 2*m + q: d log-spaced 0.5..20 over m = 0..B/2-1, alpha = 1e-4 (q=0) or 1e-3 (q=1)
        m = np.arange(B) // 2
        q = np.arange(B) % 2
        nm = max(B // 2 - 1, 1)
        d_ = 0.5 * 40.0 ** (m / nm)
        al_ = np.where(q == 0, 1e-4, 1e-3)
        r_, _, _, cr_ = _scalars(B, 1.0, 0.0, 0.0, 1.0)
        st = 5000 if steps is None else steps
        name = f"cfg4 batched sweep {B}x{nx}x{ny}"
    else:
        raise ValueError(f"unknown config {cfg}")

    dt = dt_rule(h, float(np.max(al_)), a, b, c)
    dtypes = ("f64", "f32") if cfg == 3 else ("f64",)
    return Workload(name=name, cfg=cfg, nx=nx, ny=ny, h=h, batch=B, r=r_, d=d_, alpha=al_,
                    c_r=cr_, a=a, b=b, c=c, U=U, V=V, W=W, dt=dt, steps=st, dtypes=dtypes)


def random_problem(seed: int, nx: int, ny: int, *, batch: int = 1, hetero: bool = True,
                   bmax: float = 0.8, dy_ratio: float = 1.0):
    """Generic seeded smooth-ish random problem for parity tests on odd shapes: positive-definite
    tensor with |b| <= bmax*sqrt(a*c), state in [0,1].  Pure input construction."""
    rng = np.random.default_rng([SEED, 99, seed])
    h = H
    if hetero:
        a = rng.uniform(5e-3, 2e-2, (ny, nx))
        c = rng.uniform(5e-3, 2e-2, (ny, nx))
        b = rng.uniform(-bmax, bmax, (ny, nx)) * np.sqrt(a * c)
    else:
        a = np.full((ny, nx), 1.2e-2)
        c = np.full((ny, nx), 7e-3)
        b = np.full((ny, nx), bmax * np.sqrt(1.2e-2 * 7e-3))
    U = rng.uniform(0.0, 1.0, (batch, ny, nx))
    V = rng.uniform(0.0, 1.0, (batch, ny, nx))
    W = rng.uniform(0.0, 1.0, (batch, ny, nx))
    r_ = rng.uniform(0.5, 1.5, batch)
    d_ = rng.uniform(0.5, 12.0, batch)
    al_ = rng.uniform(1e-4, 2e-3, batch)
    cr_ = rng.uniform(0.5, 2.0, batch)
    hy = h * dy_ratio                      # dy = dy_ratio * dx
    dt = dt_rule(min(h, hy), float(al_.max()), a, b, c)
    return Workload(name=f"random {batch}x{nx}x{ny} seed {seed}", cfg=-1, nx=nx, ny=ny, h=h,
                    batch=batch, r=r_, d=d_, alpha=al_, c_r=cr_, a=a, b=b, c=c, U=U, V=V, W=W,
                    dt=dt, steps=8, hy=None if dy_ratio == 1.0 else hy)


# ---------------------------------------------------------------------------------------------
# Three-dimensional extension.  The paper prints no 3-D
# experiment; the recipe carries config 2's into a box: a smooth heterogeneous positive-definite
# tensor built from seeded cosine modes, a tumour BALL in healthy tissue, no acid.  Input
# construction only (the step-size rule is the one arithmetic exception, as in 2-D).
# ---------------------------------------------------------------------------------------------
@dataclass
class Workload3:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    r: float
    d: float
    alpha: float
    c_r: float
    tensor: tuple        # (axx, ayy, azz, axy, axz, ayz), each [nz][ny][nx]
    U: np.ndarray        # [nz][ny][nx]
    V: np.ndarray
    W: np.ndarray
    dt: float
    steps: int

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


def dt_rule3(hmin: float, alpha: float, tensor) -> float:
    """0.12 * hmin^2 / max(alpha, max over cells of the largest absolute row sum of A) -- Gershgorin's
    bound on lambda_max(A); 0.12 < 1/6 keeps the seven-point diagonal part monotone in 3-D."""
    axx, ayy, azz, axy, axz, ayz = tensor
    rows = np.maximum(np.maximum(axx + np.abs(axy) + np.abs(axz), ayy + np.abs(axy) + np.abs(ayz)),
                      azz + np.abs(axz) + np.abs(ayz))
    return 0.12 * hmin * hmin / max(alpha, float(rows.max()))


def _modes3(rng, x, y, z, L):
    """a field in [-1, 1] from 6 seeded cosine modes with wavenumbers 1..3 over the box:
    cos(tx + ty + tz + ph) assembled from an xy-plane factor and a z factor (one pass per mode)"""
    f = np.zeros(np.broadcast_shapes(x.shape, y.shape, z.shape))
    for _ in range(6):
        kx, ky, kz = rng.integers(1, 4, 3)
        ph = rng.uniform(0.0, 2.0 * np.pi)
        txy = 2.0 * np.pi * (kx * x / L[0] + ky * y / L[1])          # [1][ny][nx]
        tz = 2.0 * np.pi * kz * z / L[2] + ph                         # [nz][1][1]
        f += np.cos(txy) * np.cos(tz)
        f -= np.sin(txy) * np.sin(tz)
    f /= 6.0
    return f


def make3d(nx: int, ny: int, nz: int, *, steps: int = 10, d: float = 10.0, seed: int = 0,
           spacing=(H, H, H), random_state: bool = False) -> Workload3:
    """Seeded 3-D problem: diagonal entries 1e-2 (1 + f/2), off-diagonals 0.3 g sqrt(a_pp a_qq)
    (|0.3 g| <= 0.3 on all three keeps A positive definite by Gershgorin), a tumour ball of radius
    0.12 L centred at (0.4, 0.55, 0.5) L with V = 1, U = 0 inside, U = 1, V = 0 outside, W = 0, plus
    uniform [0, 1e-3) noise on U then V, clipped.  random_state: uniform [0,1) fields instead (parity
    tests on tiny or awkward shapes)."""
    rng = np.random.default_rng([SEED, 3, nx, ny, nz, seed])
    dx, dy, dz = spacing
    L = (nx * dx, ny * dy, nz * dz)
    x = ((np.arange(nx) + 0.5) * dx)[None, None, :]
    y = ((np.arange(ny) + 0.5) * dy)[None, :, None]
    z = ((np.arange(nz) + 0.5) * dz)[:, None, None]
    diag = [1e-2 * (1.0 + 0.5 * _modes3(rng, x, y, z, L)) for _ in range(3)]
    g = [_modes3(rng, x, y, z, L) for _ in range(3)]
    axy = 0.3 * g[0] * np.sqrt(diag[0] * diag[1])
    axz = 0.3 * g[1] * np.sqrt(diag[0] * diag[2])
    ayz = 0.3 * g[2] * np.sqrt(diag[1] * diag[2])
    tensor = tuple(np.ascontiguousarray(t) for t in (*diag, axy, axz, ayz))
    shape = (nz, ny, nx)
    if random_state:
        U, V, W = (rng.uniform(0.0, 1.0, shape) for _ in range(3))
    else:
        rad = 0.12 * min(L)
        inside = (x - 0.4 * L[0]) ** 2 + (y - 0.55 * L[1]) ** 2 + (z - 0.5 * L[2]) ** 2 <= rad * rad
        U = np.where(inside, 0.0, 1.0) + rng.uniform(0.0, 1e-3, shape)
        V = np.where(inside, 1.0, 0.0) + rng.uniform(0.0, 1e-3, shape)
        U, V, W = np.clip(U, 0.0, 1.0), np.clip(V, 0.0, 1.0), np.zeros(shape)
    alpha = 1e-3
    return Workload3(name=f"3-D smooth heterogeneous {nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz,
                     r=1.0, d=d, alpha=alpha, c_r=1.0, tensor=tensor, U=U, V=V, W=W,
                     dt=dt_rule3(min(spacing), alpha, tensor), steps=steps)
