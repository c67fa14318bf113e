"""Full-size parity (-m gpu): BASELINE.json's headline sizes in the launch configuration that
bench.py times (default kernel selection, graphs on), checked on sampled outputs.

The oracle cannot afford 8192^2 x many steps, so each sampled window is cut out of the inputs with
a margin of n cells on its interior sides (the stencils move information one cell per step), the
oracle runs n steps on the cut, and the uncontaminated core is compared element by element.
Windows sit where the kernel's decomposition has seams: domain corners and edges (Neumann faces),
strip / tile-column boundaries (x = 64, 512 cells), row-chunk boundaries, tensor band
discontinuities and tumour fronts.  Plus properties that hold at any size.
"""
import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-10, "f32": 2e-4}
WIN = 40


def check_windows(wl, sim_idx, got, n, spots, dtype):
    """spots: (i0, j0) for a WIN x WIN window or (i0, j0, wx, wy)."""
    worst = 0.0
    for spot in spots:
        i0, j0 = spot[:2]
        wx, wy = spot[2:] if len(spot) == 4 else (WIN, WIN)
        i0 = int(min(max(i0, 0), wl.nx - wx))
        j0 = int(min(max(j0, 0), wl.ny - wy))
        ia, ja = max(i0 - n, 0), max(j0 - n, 0)
        ib, jb = min(i0 + wx + n, wl.nx), min(j0 + wy + n, wl.ny)
        cut = (slice(ja, jb), slice(ia, ib))
        s = sim_idx
        ref = oracle.step(wl.U[s][cut], wl.V[s][cut], wl.W[s][cut], wl.a[cut], wl.b[cut], wl.c[cut],
                          r=wl.r[s], d=wl.d[s], alpha=wl.alpha[s], c_r=wl.c_r[s], n=n, dt=wl.dt,
                          dx=wl.h)
        core = (slice(j0 - ja, j0 - ja + wy), slice(i0 - ia, i0 - ia + wx))
        full = (slice(j0, j0 + wy), slice(i0, i0 + wx))
        for f, name in enumerate("UVW"):
            err = float(np.max(np.abs(got[f][s][full].astype(np.float64) - ref[f][core])))
            assert err <= TOL[dtype], f"window ({i0},{j0}) sim {s} field {name}: {err:.3e}"
            worst = max(worst, err)
    return worst


@pytest.fixture(scope="module")
def cfg3():
    return workloads.make(3)


def seam_spots(wl):
    nx, ny = wl.nx, wl.ny
    band = ny // 6
    jj, ii = np.nonzero(wl.V[0] > 0.5)
    k = int(np.argmin(ii))
    front = (int(ii[k]) - WIN // 2, int(jj[k]) - WIN // 2)
    return [(0, 0), (nx - WIN, 0), (0, ny - WIN), (nx - WIN, ny - WIN),      # corners
            (512 - WIN // 2, band - WIN // 2),                               # tile seam x band jump
            (64 - WIN // 2, 222 - WIN // 2), (4096 - WIN // 2, 2 * band - WIN // 2),
            (nx - WIN, 5 * band - WIN // 2), (1024 - WIN // 2, 221), front,
            # a full-height strip across a tile-column seam: crosses EVERY row-chunk boundary of
            # whatever plan the library picked; a full-width strip: crosses every tile column
            (236 - 12, 0, 24, ny), (0, 3 * band - 12, nx, 24)]


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config3_full_size_sampled(cfg3, dtype):
    wl, n = cfg3, 7      # one four-step, one two-step and one single-step launch
    with binding.from_workload(wl, dtype=dtype) as sim:
        # what AUTO resolves to, i.e. what bench.py times: four steps per launch in both types
        assert sim.kernel == "quad"
        sim.step(n, wl.dt)
        assert sim.launches == n // 4 + (n % 4) // 2 + n % 2
        got = sim.get_state_numpy()
    for g in got:
        assert np.isfinite(g).all()
    worst = check_windows(wl, 0, got, n, seam_spots(wl), dtype)
    print(f"cfg3 {dtype} full size: worst window error {worst:.3e}")


def test_config3_full_size_conservation_and_bounds(cfg3):
    """Any-size properties on the GPU result: with r = c_r = 0, sum V and sum W are conserved
    (zero-flux boundaries, reading A2)."""
    import torch
    wl = cfg3
    with binding.Simulation(wl.nx, wl.ny, wl.h, 0.0, wl.d, wl.alpha, 0.0) as sim:
        sim.set_tensor(wl.a, wl.b, wl.c)
        sim.set_state(wl.U, wl.V, wl.V)          # W0 := V0 so that sum W is not trivially 0
        sim.step(8, wl.dt)
        U, V, W = sim.get_state()
        sV, sW = float(V.sum()), float(W.sum())
        s0 = float(np.sum(wl.V, dtype=np.float64))
        assert abs(sV - s0) <= 1e-11 * s0
        assert abs(sW - s0) <= 1e-11 * s0
        assert bool(torch.isfinite(U).all()) and bool(torch.isfinite(W).all())


def test_config4_full_size_batch_sampled():
    wl = workloads.make(4)
    assert wl.batch == 64 and wl.nx == 1024
    n = 5
    with binding.from_workload(wl) as sim:
        sim.step(n, wl.dt)
        got = sim.get_state_numpy()
    jj, ii = np.nonzero(wl.V[0] > 0.5)
    k = int(np.argmin(jj))
    spots = [(0, 0), (wl.nx - WIN, wl.ny - WIN), (512 - WIN // 2, 300),
             (int(ii[k]) - WIN // 2, int(jj[k]) - WIN // 2)]
    for s in (0, 1, 31, 32, 63):
        check_windows(wl, s, got, n, spots, "f64")
    # simulations with different d must have diverged from one another
    assert np.max(np.abs(got[0][0] - got[0][62])) > 1e-6


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_large_ragged_grid_sampled(dtype):
    """A grid wider than the headline one in cells per row for fp32 tiles, ragged against every
    tile width of the library (236 / 480 / 944 / 1888 cells) and against the row chunks: 10008 x
    5001 cells, AUTO kernel, six steps (one four-step + one two-step launch)."""
    wl = workloads.make(3, nx=10008, ny=5001)
    n = 6
    with binding.from_workload(wl, dtype=dtype) as sim:
        assert sim.kernel == "quad"
        sim.step(n, wl.dt)
        got = sim.get_state_numpy()
    for g in got:
        assert np.isfinite(g).all()
    nx, ny = wl.nx, wl.ny
    spots = [(0, 0), (nx - WIN, 0), (0, ny - WIN), (nx - WIN, ny - WIN),
             (nx - 24, 0, 24, ny),            # the ragged last tile column, every row chunk
             (0, ny - 24, nx, 24),            # the top rows, every tile column
             (9912 - 12, 2500, 24, 200)]      # 42 x 236: the last full four-step tile seam
    check_windows(wl, 0, got, n, spots, dtype)
