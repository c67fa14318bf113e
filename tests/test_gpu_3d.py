"""GPU parity of the three-dimensional extension (include/gg3.h) against the 3-D oracle, through the
C ABI: both kernels, both dtypes, ragged tiles and z chunks, dx != dy != dz, every Neumann face,
edge and corner, equilibria, mass conservation; the two kernels bit-identical to each other.
Tolerances: north_star's (fp64 1e-10, fp32 2e-4 max-abs per field)."""
import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, binding3, workloads

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-10, "f32": 2e-4}
KERNELS = {"generic": binding3.GG3_KERNEL_GENERIC, "tiled": binding3.GG3_KERNEL_TILED}


def oracle_run(wl, n):
    return oracle.step3d(wl.U, wl.V, wl.W, wl.tensor, r=wl.r, d=wl.d, alpha=wl.alpha, c_r=wl.c_r, n=n,
                         dt=wl.dt, dx=wl.dx, dy=wl.dy, dz=wl.dz)


def gpu_run(wl, n, dtype="f64", kernel=None, split=None):
    with binding3.from_workload(wl, dtype=dtype) as sim:
        if kernel is not None:
            sim.set_option(binding3.GG3_OPT_KERNEL, KERNELS[kernel])
        for m in (split or [n]):
            sim.step(m, wl.dt)
        assert sim.launches == n
        return sim.get_state_numpy(), sim.kernel


def assert_close(got, ref, dtype, what):
    for name, g, r in zip("UVW", got, ref):
        assert g.shape == r.shape and np.isfinite(g).all(), f"{what}: {name}"
        err = float(np.max(np.abs(g.astype(np.float64) - r)))
        assert err <= TOL[dtype], f"{what}: field {name} max-abs error {err:.3e} > {TOL[dtype]:.0e}"


@pytest.mark.parametrize("kernel", ["generic", "tiled"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_shapes_and_boundaries(kernel, dtype):
    # 2^3 (every cell a corner), one tile, ragged tiles in x and y, several z chunks, thin slabs
    for nx, ny, nz in ((2, 2, 2), (3, 2, 5), (32, 8, 4), (33, 9, 17), (70, 21, 40), (5, 37, 3), (96, 50, 9)):
        wl = workloads.make3d(nx, ny, nz, random_state=True, seed=nx)
        for n in (1, 6):
            got, used = gpu_run(wl, n, dtype=dtype, kernel=kernel)
            assert used == kernel
            assert_close(got, oracle_run(wl, n), dtype, f"{kernel} {dtype} {nx}x{ny}x{nz} n={n}")


def test_config_recipe_long_run_and_kernels_bit_identical():
    wl = workloads.make3d(72, 40, 36, steps=120)
    ref = oracle_run(wl, wl.steps)
    a, ka = gpu_run(wl, wl.steps, kernel="tiled", split=[1, 7, wl.steps - 8])
    b, kb = gpu_run(wl, wl.steps, kernel="generic")
    assert (ka, kb) == ("tiled", "generic")
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert_close(a, ref, "f64", "3-D recipe, 120 steps")
    got32, _ = gpu_run(wl, wl.steps, dtype="f32")
    assert_close(got32, ref, "f32", "3-D recipe, 120 steps, fp32")
    # the tumour ball has spread and made acid: the run is not vacuous
    assert ref[2].max() > 0.05 and ref[0].min() < 0.5


def test_graph_replay_is_bit_identical_to_plain_launches_and_caches_by_dt():
    """gg3_step replays cached CUDA graphs (GG3_OPT_GRAPH, default on).  Odd and even chunk
    lengths, a ragged last chunk, split calls: the end state equals the plain-launch loop bit for
    bit; a loop with one dt captures each (length, parity) once, a second dt captures anew (the 3-D
    kernels take their coefficients by value)."""
    wl = workloads.make3d(70, 21, 24, steps=37, random_state=True)
    with binding3.from_workload(wl) as sim:
        sim.set_option(binding3.GG3_OPT_GRAPH, 0)
        sim.step(wl.steps, wl.dt)
        sim.step(5, 0.5 * wl.dt)
        plain = sim.get_state_numpy()
        assert sim.graph_captures == 0 and sim.launches == 42
    with binding3.from_workload(wl) as sim:
        sim.set_option(binding3.GG3_OPT_GRAPH_CHUNK, 7)       # 37 = 5 x 7 + 2: parities alternate
        sim.step(wl.steps, wl.dt)
        caps = sim.graph_captures
        assert caps == 3                                      # (7, parity 0), (7, parity 1), (2, parity 1)
        sim.step(5, 0.5 * wl.dt)                              # new dt: one more capture
        assert sim.graph_captures == caps + 1 and sim.launches == 42
        graph = sim.get_state_numpy()
        sim.step(5, 0.5 * wl.dt)                              # same key, other parity
        sim.step(5, 0.5 * wl.dt)                              # cached
        assert sim.graph_captures == caps + 2
    for x, y in zip(plain, graph):
        assert np.array_equal(x, y)
    assert_close(graph, oracle.step3d(*oracle_run(wl, wl.steps), wl.tensor, r=wl.r, d=wl.d, alpha=wl.alpha,
                                      c_r=wl.c_r, n=5, dt=0.5 * wl.dt, dx=wl.dx, dy=wl.dy, dz=wl.dz),
                 "f64", "graph replay, two step sizes")


def test_anisotropic_mesh():
    wl = workloads.make3d(40, 24, 20, spacing=(1 / 64, 1 / 48, 1 / 80), random_state=True)
    for kernel in ("generic", "tiled"):
        got, _ = gpu_run(wl, 25, kernel=kernel)
        assert_close(got, oracle_run(wl, 25), "f64", f"dx != dy != dz {kernel}")


def test_auto_picks_the_tiled_kernel_and_equilibria_are_exact():
    wl = workloads.make3d(48, 20, 12)
    for state in ((1.0, 0.0, 0.0), (0.0, 1.0, 1.0), (0.0, 0.0, 0.0)):
        wl.U, wl.V, wl.W = (np.full((wl.nz, wl.ny, wl.nx), s) for s in state)
        got, used = gpu_run(wl, 9)
        assert used == "tiled"
        for g, s in zip(got, state):
            assert np.all(g == s)


def test_mass_conservation_without_reactions():
    wl = workloads.make3d(50, 30, 22, random_state=True)
    wl.r, wl.d, wl.c_r = 0.0, 0.0, 0.0
    got, _ = gpu_run(wl, 40)
    assert abs(got[2].sum() - wl.W.sum()) <= 1e-12 * wl.W.sum()
    assert abs(got[1].sum() - wl.V.sum()) <= 1e-12 * wl.V.sum()


def test_errors():
    with pytest.raises(binding.GGError) as e:
        binding3.gg3_create(1, 4, 4, 1.0, 1.0, 1.0, 1.0, 1.0, 1e-3, 1.0)
    assert e.value.code == binding.GG_ERR_ARG
    wl = workloads.make3d(8, 8, 8)
    with binding3.from_workload(wl) as sim:
        with pytest.raises(binding.GGError):
            sim.step(1, -1.0)
        with pytest.raises(binding.GGError):
            sim.set_option(7, 0)
