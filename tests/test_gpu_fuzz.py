"""Bounded random-shape fuzz (-m gpu, fixed seed, ~20 s): every kernel of libgg through the C ABI
against the CPU oracle AND against the one-thread-per-cell kernel bit for bit.  Shapes are drawn
around the kernels' tile widths (60, 118, 236, 240, 472, 480, 944 cells), tiny and ragged heights,
batches, odd step counts and dx != dy."""
import time

import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding as B, workloads

pytestmark = pytest.mark.gpu
KERNELS = {"generic": B.GG_KERNEL_GENERIC, "stream": B.GG_KERNEL_STREAM, "stream2": B.GG_KERNEL_STREAM2,
           "resident": B.GG_KERNEL_RESIDENT, "pair": B.GG_KERNEL_PAIR, "quad": B.GG_KERNEL_QUAD}


def test_fuzz_all_kernels_bounded():
    rng = np.random.default_rng(20060174)
    t0, ncase = time.time(), 0
    while time.time() - t0 < 20.0 or ncase < 12:
        dtype = str(rng.choice(["f64", "f32"]))
        c = 2 if dtype == "f64" else 4
        nx = int(rng.choice([c, 2 * c, 60, 59 * c, 236, 240, 472, 480, 944, int(rng.integers(1, 700)) * c]))
        ny = int(rng.choice([2, 3, 4, 5, 7, 8, 15, 16, 17, 31, 33, 64, int(rng.integers(2, 400))]))
        batch = int(rng.choice([1, 1, 2, 3, 5]))
        if nx * ny * batch > 600000:
            continue
        n = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 9, 12, 13]))
        ratio = float(rng.choice([1.0, 1.0, 0.5, 1.6]))
        wl = workloads.random_problem(int(rng.integers(1 << 30)), nx, ny, batch=batch, dy_ratio=ratio)
        ref = [oracle.step(wl.U[s], wl.V[s], wl.W[s], wl.a, wl.b, wl.c, r=wl.r[s], d=wl.d[s],
                           alpha=wl.alpha[s], c_r=wl.c_r[s], n=n, dt=wl.dt, dx=wl.h, dy=wl.dy)
               for s in range(batch)]
        outs = {}
        for name, k in KERNELS.items():
            try:
                with B.from_workload(wl, dtype=dtype) as sim:
                    sim.set_option(B.GG_OPT_KERNEL, k)
                    sim.step(n, wl.dt)
                    outs[name] = sim.get_state_numpy()
            except B.GGError as e:
                if e.code != B.GG_ERR_UNSUPPORTED:   # a shape the kernel declares it cannot take
                    raise
        tol = 1e-10 if dtype == "f64" else 2e-4
        for name, got in outs.items():
            err = max(float(np.max(np.abs(got[f][s].astype(np.float64) - ref[s][f])))
                      for f in range(3) for s in range(batch))
            assert err <= tol, (dtype, nx, ny, batch, n, ratio, name, err)
            assert all(np.array_equal(got[f], outs["generic"][f]) for f in range(3)), \
                (dtype, nx, ny, batch, n, ratio, name, "differs from generic")
        ncase += 1
    print(f"fuzz: {ncase} cases")


def test_onchip_kernels_many_calls_bit_identical():
    """The on-chip kernels (one cluster per simulation with st.async halo rows where it fits, row
    slabs otherwise) over calls of 1, 7, 64 and 301 steps on random small shapes and batches, bit
    for bit against the single-step kernel: a lost or early halo hand-off changes bits."""
    rng = np.random.default_rng(5)
    ncase = 0
    for it in range(16):
        nx = int(rng.choice([8, 16, 32, 64, 96, 128, 160]))
        ny = int(rng.integers(2, 150))
        b = int(rng.choice([1, 1, 2, 5, 9, 20]))
        dtype = str(rng.choice(["f64", "f32"]))
        wl = workloads.random_problem(1000 + it, nx, ny, batch=b)
        outs = []
        for kern in ("resident", "stream"):
            with B.from_workload(wl, dtype=dtype) as sim:
                try:
                    sim.set_option(B.GG_OPT_KERNEL, KERNELS[kern])
                except B.GGError:
                    outs = None
                    break
                for n in (1, 7, 64, 301):
                    sim.step(n, wl.dt)
                outs.append(sim.get_state_numpy())
        if outs is None:
            continue
        ncase += 1
        for x, y in zip(*outs):
            assert np.array_equal(x, y), f"on-chip kernel differs from stream: {nx}x{ny}x{b} {dtype}"
    assert ncase >= 8


def test_cluster_kernel_stress_thin_slabs_long_calls_many_clusters():
    """The cluster kernel's halo protocol (remote st.async rows completed on the receiver's
    mbarrier, two state copies reused every second step on the argument that a neighbour is at most
    one step ahead) where it is most exposed: ONE row per CTA and grids with fewer rows than the
    cluster has CTAs (some CTAs own nothing), both cluster sizes, batches of 40 and 75 simulations
    (more clusters than the GPU holds at once, so waves of clusters start and finish at different
    times), and thousands of steps inside a single launch.  Bit for bit against the single-step
    kernel: a hand-off that is lost, early or late changes bits."""
    cases = [  # nx, ny, batch, dtype, cluster CTAs (0 = the library's choice), steps per call
        (32, 16, 1, "f64", 16, (3000, 1)),     # R = 1 with every CTA busy
        (64, 5, 40, "f64", 8, (1501, 2)),      # ny < CL: three CTAs of every cluster own no row
        (16, 2, 75, "f32", 16, (2000,)),       # two rows in a 16-CTA cluster, 75 clusters
        (128, 9, 40, "f32", 8, (999, 64)),     # R = 2, the last CTAs ragged / empty
        (96, 33, 9, "f64", 0, (1200, 7)),
    ]
    for nx, ny, b, dtype, ctas, calls in cases:
        wl = workloads.random_problem(7000 + nx + ny, nx, ny, batch=b)
        outs = []
        for kern in ("resident", "stream"):
            with B.from_workload(wl, dtype=dtype) as sim:
                sim.set_option(B.GG_OPT_KERNEL, KERNELS[kern])
                if kern == "resident" and ctas:
                    sim.set_option(B.GG_OPT_CLUSTER_CTAS, ctas)
                for n in calls:
                    sim.step(n, wl.dt)
                    if kern == "resident":
                        assert "gg_step_cluster" in sim.kernel_name, sim.kernel_name
                outs.append(sim.get_state_numpy())
        for x, y in zip(*outs):
            assert np.isfinite(x).all()
            assert np.array_equal(x, y), f"cluster kernel differs from stream: {nx}x{ny}x{b} {dtype} CL={ctas}"
