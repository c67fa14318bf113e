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
