"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle,
element by element on the same seeded inputs.

Tolerances (BASELINE.json north_star): fp64 max-abs 1e-10 per field, fp32
storage 2e-4, after the stated step count.  The oracle always runs in fp64 from the fp64 inputs;
the fp32 GPU path gets the same arrays rounded to nearest fp32 (reading A10).
"""
import numpy as np
import pytest

import oracle
from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-10, "f32": 2e-4}
KERNELS = {"generic": binding.GG_KERNEL_GENERIC, "stream": binding.GG_KERNEL_STREAM,
           "stream2": binding.GG_KERNEL_STREAM2, "pair": binding.GG_KERNEL_PAIR,
           "quad": binding.GG_KERNEL_QUAD, "resident": binding.GG_KERNEL_RESIDENT}


def expected_launches(kernel, calls, explicit=True, min_steps=8):
    """Kernel launches for a list of gg_step(n) calls: stream2 / pair advance two steps per launch,
    quad four (then two, then one), resident all n steps of a call (under AUTO only for calls of
    at least `min_steps` steps -- 4 for the cluster kernel, 8 for the slab kernel; shorter ones run
    stream2)."""
    two = lambda n: n // 2 + n % 2
    if kernel == "resident":
        return sum((1 if n > 0 else 0) if (explicit or n >= min_steps) else two(n) for n in calls)
    if kernel == "quad":
        return sum(n // 4 + (n % 4) // 2 + n % 2 for n in calls)
    if kernel in ("stream2", "pair"):
        return sum(two(n) for n in calls)
    return sum(calls)


def oracle_run(wl, steps):
    outs = [oracle.step(wl.U[s], wl.V[s], wl.W[s], wl.a, wl.b, wl.c, r=wl.r[s], d=wl.d[s],
                        alpha=wl.alpha[s], c_r=wl.c_r[s], n=steps, dt=wl.dt, dx=wl.h, dy=wl.dy)
            for s in range(wl.batch)]
    return tuple(np.stack([o[f] for o in outs]) for f in range(3))


def gpu_run(wl, steps, dtype="f64", kernel=None, options=(), split=None, check_launches=True):
    with binding.from_workload(wl, dtype=dtype) as sim:
        if kernel is not None:
            sim.set_option(binding.GG_OPT_KERNEL, KERNELS[kernel])
        for opt, val in options:
            sim.set_option(opt, val)
        for n in (split or [steps]):
            sim.step(n, wl.dt)
        used = sim.kernel
        min_steps = 4 if "cluster" in sim.kernel_name else 8
        launches = sim.launches
        out = sim.get_state_numpy()
    if check_launches:   # (graph chunks shorter than a call split it like separate calls)
        assert launches == expected_launches(used, split or [steps], explicit=kernel is not None, min_steps=min_steps)
    return out, used


def assert_close(got, ref, dtype, what=""):
    for name, g, r in zip("UVW", got, ref):
        assert g.shape == r.shape
        assert np.isfinite(g).all(), f"{what}: non-finite {name}"
        err = float(np.max(np.abs(g.astype(np.float64) - r)))
        assert err <= TOL[dtype], f"{what}: field {name} max-abs error {err:.3e} > {TOL[dtype]:.0e}"


# ---------------------------------------------------------------------------------------------
# BASELINE.json configs (0 and 1 at full size and step count; 2-4 at oracle-sized grids with the
# same recipe, ragged in both directions so that strips, chunks and TMA boxes have partial tails)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", ["stream", "stream2", "generic"])
def test_config0_full(kernel):
    wl = workloads.make(0)
    got, used = gpu_run(wl, wl.steps, kernel=kernel)
    assert used == kernel
    assert_close(got, oracle_run(wl, wl.steps), "f64", f"cfg0 {kernel}")


def test_config1_full():
    wl = workloads.make(1)
    got, used = gpu_run(wl, wl.steps)
    assert used == "quad"      # AUTO: mid-size fp64 grids run four steps per launch
    ref = oracle_run(wl, wl.steps)
    assert_close(got, ref, "f64", "cfg1")


def test_config1_undershoot_is_reproduced_not_repaired():
    """Reading A7: with b != 0 the scheme drives W slightly below 0 (and then U above 1) early in
    the run; the GPU must show the same values as the oracle, never a clamped field."""
    wl = workloads.make(1)
    got, _ = gpu_run(wl, 6)
    ref = oracle_run(wl, 6)
    assert ref[2].min() < -1e-5 and ref[0].max() > 1.0
    assert got[2].min() < -1e-5 and got[0].max() > 1.0
    assert_close(got, ref, "f64", "cfg1 after 6 steps")


@pytest.mark.parametrize("d", [2.0, 10.0, 20.0])
def test_config2_reduced_d_sweep(d):
    wl = workloads.make(2, nx=328, ny=203, steps=400, d=d)
    got, _ = gpu_run(wl, wl.steps)
    assert_close(got, oracle_run(wl, wl.steps), "f64", f"cfg2 d={d}")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("kernel", ["stream", "stream2", "generic"])
def test_config3_reduced_banded(dtype, kernel):
    wl = workloads.make(3, nx=392, ny=250, steps=300)
    got, _ = gpu_run(wl, wl.steps, dtype=dtype, kernel=kernel)
    assert_close(got, oracle_run(wl, wl.steps), dtype, f"cfg3 {dtype} {kernel}")


def test_config4_reduced_batch():
    wl = workloads.make(4, nx=136, ny=90, batch=6, steps=250)
    assert len(set(wl.d)) > 1 and len(set(wl.alpha)) > 1
    got, _ = gpu_run(wl, wl.steps)
    assert_close(got, oracle_run(wl, wl.steps), "f64", "cfg4")


# ---------------------------------------------------------------------------------------------
# random problems on awkward shapes, every kernel and every tuned build of the stream kernel
# ---------------------------------------------------------------------------------------------
SHAPES = [(2, 2), (2, 7), (4, 2), (64, 5), (66, 37), (130, 3), (258, 71), (62, 129)]


@pytest.mark.parametrize("nx,ny", SHAPES)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_random_shapes(nx, ny, dtype):
    wl = workloads.random_problem(nx * 1000 + ny, nx, ny)
    ref = oracle_run(wl, 9)
    kernels = ["generic"]
    if (nx * (8 if dtype == "f64" else 4)) % 16 == 0:
        kernels += ["stream", "stream2"]
    for kernel in kernels:
        got, used = gpu_run(wl, 9, dtype=dtype, kernel=kernel)
        assert used == kernel
        assert_close(got, ref, dtype, f"{nx}x{ny} {dtype} {kernel}")


@pytest.mark.parametrize("nx,ny", [(65, 9), (3, 3), (127, 33)])
def test_odd_width_takes_generic_path(nx, ny):
    wl = workloads.random_problem(7 + nx, nx, ny)
    got, used = gpu_run(wl, 5)
    assert used == "generic"  # AUTO never mis-computes: rows are not 16-byte multiples
    assert_close(got, oracle_run(wl, 5), "f64", f"{nx}x{ny}")


def test_every_stream_variant_and_chunking():
    wl = workloads.random_problem(42, 328, 150, batch=2)   # 6 strips: ragged tile columns
    ref = oracle_run(wl, 7)
    for v in range(binding.gg_num_stream_variants()):
        for nw in (0, 1, 2, 4, 8):
            for ipc in (1, 64):
                got, _ = gpu_run(wl, 7, kernel="stream",
                                 options=[(binding.GG_OPT_STREAM_VARIANT, v),
                                          (binding.GG_OPT_STREAM_WARPS, nw),
                                          (binding.GG_OPT_ITEMS_PER_WARP, ipc)])
                assert_close(got, ref, "f64", f"variant {v} warps {nw} items/CTA {ipc}")


def test_wide_grid_fp32_and_fp64_all_warp_counts():
    """1100 fp32 / 1030 fp64 cells per row: several full tile columns plus a ragged last one."""
    for dtype, nx in (("f32", 1100), ("f64", 1030)):
        wl = workloads.random_problem(77, nx, 45)
        ref = oracle_run(wl, 5)
        for nw in (1, 2, 4, 8):
            got, _ = gpu_run(wl, 5, dtype=dtype, kernel="stream",
                             options=[(binding.GG_OPT_STREAM_WARPS, nw)])
            assert_close(got, ref, dtype, f"{dtype} nx={nx} warps {nw}")


def test_every_stream2_variant_warps_and_chunking():
    wl = workloads.random_problem(43, 328, 150, batch=2)   # 6 strips: ragged tile columns
    ref = {n: oracle_run(wl, n) for n in (6, 7)}
    for v in range(binding.gg_num_stream2_variants()):
        for nw in (0, 1, 2, 4):
            for ipc, n in ((1, 7), (64, 6)):
                got, used = gpu_run(wl, n, kernel="stream2",
                                    options=[(binding.GG_OPT_STREAM2_VARIANT, v),
                                             (binding.GG_OPT_STREAM_WARPS, nw),
                                             (binding.GG_OPT_ITEMS_PER_WARP, ipc)])
                assert used == "stream2"
                assert_close(got, ref[n], "f64", f"stream2 variant {v} warps {nw} items/CTA {ipc}")


def test_stream2_wide_ragged_fp32_fp64():
    for dtype, nx in (("f32", 1100), ("f64", 1030)):
        wl = workloads.random_problem(78, nx, 45)
        ref = oracle_run(wl, 6)
        for nw in (1, 2, 4):
            got, _ = gpu_run(wl, 6, dtype=dtype, kernel="stream2",
                             options=[(binding.GG_OPT_STREAM_WARPS, nw)])
            assert_close(got, ref, dtype, f"stream2 {dtype} nx={nx} warps {nw}")


def test_stream2_equals_two_single_steps():
    """The two-step kernel applies the single-step march twice: same arithmetic, same order."""
    wl = workloads.make(2, nx=520, ny=300, steps=40)
    a, _ = gpu_run(wl, 40, kernel="stream2")
    b, _ = gpu_run(wl, 40, kernel="stream")
    c, _ = gpu_run(wl, 40, kernel="generic")
    for x, y, z in zip(a, b, c):
        assert np.array_equal(x, y)     # bit-identical: explicit rounding points (gg_common.cuh)
        assert np.array_equal(x, z)
    assert_close(a, oracle_run(wl, 40), "f64", "stream2 cfg2")


def test_stream2_config4_batch_and_split_calls():
    wl = workloads.make(4, nx=264, ny=90, batch=5, steps=60)
    got, _ = gpu_run(wl, 60, kernel="stream2", split=[1, 2, 3, 0, 7, 47])
    assert_close(got, oracle_run(wl, 60), "f64", "stream2 cfg4 split")


def test_stream_and_generic_agree_closely():
    """Two independent kernels inside the library: same scheme, different evaluation order."""
    wl = workloads.random_problem(5, 192, 96)
    a, _ = gpu_run(wl, 50, kernel="stream")
    b, _ = gpu_run(wl, 50, kernel="generic")
    for x, y in zip(a, b):
        assert np.max(np.abs(x - y)) < 1e-12


# ---------------------------------------------------------------------------------------------
# step loop: graphs, ping-pong parity, repeated calls
# ---------------------------------------------------------------------------------------------
def test_graph_and_plain_launches_give_identical_bits():
    """Graph replay (odd chunk lengths, so graphs of 4-, 2- and 1-step launches are mixed) against
    plain launches, for every multi-launch kernel."""
    wl = workloads.make(2, nx=520, ny=120, steps=1)
    ref = None
    for kernel in ("stream", "stream2", "pair", "quad"):
        for chunk in (7, 16, 64):
            a, _ = gpu_run(wl, 131, kernel=kernel, options=[(binding.GG_OPT_GRAPH, 1), (binding.GG_OPT_GRAPH_CHUNK, chunk)],
                           check_launches=False)
            ref = a if ref is None else ref
            for x, y in zip(a, ref):
                assert np.array_equal(x, y)
        b, _ = gpu_run(wl, 131, kernel=kernel, options=[(binding.GG_OPT_GRAPH, 0)])
        for x, y in zip(b, ref):
            assert np.array_equal(x, y)
    assert_close(ref, oracle_run(wl, 131), "f64", "graph replay")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("ratio", [0.5, 1.75])
def test_rectangular_mesh_dx_ne_dy(ratio, dtype):
    """gg_create_xy: dx != dy.  Tables 1-2 carry 1/dx^2, 1/dy^2 and 1/(4 dx dy)
    separately; every kernel must weight x faces, y faces and the cross terms accordingly."""
    wl = workloads.random_problem(5, 328, 150, batch=2, dy_ratio=ratio)
    ref = oracle_run(wl, 30)
    outs = []
    for kernel in ("generic", "stream", "stream2"):
        got, used = gpu_run(wl, 30, dtype=dtype, kernel=kernel)
        assert used == kernel
        assert_close(got, ref, dtype, f"dx != dy ({ratio}) {kernel}")
        outs.append(got)
    for f in range(3):
        assert np.array_equal(outs[0][f], outs[1][f]) and np.array_equal(outs[0][f], outs[2][f])
    # and the mesh ratio matters: the square-mesh result differs
    sq = workloads.random_problem(5, 328, 150, batch=2)
    assert np.max(np.abs(oracle_run(sq, 30)[2] - ref[2])) > 1e-6


# ---------------------------------------------------------------------------------------------
# GG_KERNEL_PAIR: two steps chained in registers, x-neighbours by warp shuffle
# ---------------------------------------------------------------------------------------------
def test_pair_every_variant_warps_and_chunking():
    wl = workloads.random_problem(44, 488, 150, batch=2)   # fp64: 9 strips of 60 cells, ragged
    ref = {n: oracle_run(wl, n) for n in (2, 5)}
    base = {n: gpu_run(wl, n, kernel="stream")[0] for n in (2, 5)}
    for v in range(binding.gg_num_pair_variants()):
        for nw in (1, 3, 4, 5, 8):
            for ipc, n in ((1, 2), (4, 5), (16, 2)):
                try:
                    got, used = gpu_run(wl, n, kernel="pair",
                                        options=[(binding.GG_OPT_PAIR_VARIANT, v),
                                                 (binding.GG_OPT_STREAM_WARPS, nw),
                                                 (binding.GG_OPT_ITEMS_PER_WARP, ipc)])
                except binding.GGError as e:
                    assert e.code == binding.GG_ERR_UNSUPPORTED and "shared memory" in str(e)
                    continue
                assert used == "pair"
                assert_close(got, ref[n], "f64", f"pair variant {v} warps {nw} items/CTA {ipc}")
                for x, y in zip(got, base[n]):
                    assert np.array_equal(x, y), f"pair variant {v} warps {nw}: not bit-identical"


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_pair_shapes_dtypes_and_boundaries(dtype):
    for nx, ny, batch in ((4, 2, 1), (8, 3, 2), (60, 17, 1), (64, 64, 1), (124, 40, 3), (1000, 37, 1), (2056, 70, 1)):
        wl = workloads.random_problem(300 + nx, nx, ny, batch=batch)
        for n in (1, 2, 7):
            got, used = gpu_run(wl, n, dtype=dtype, kernel="pair")
            assert used == "pair"
            assert_close(got, oracle_run(wl, n), dtype, f"pair {dtype} {nx}x{ny}x{batch} n={n}")


def test_pair_configs_long_runs_bit_identical_to_single_step():
    for wl, n in ((workloads.make(2, nx=520, ny=300, steps=200), 200),
                  (workloads.make(3, nx=392, ny=250, steps=300), 301),
                  (workloads.make(4, nx=264, ny=90, batch=5, steps=60), 60)):
        a, _ = gpu_run(wl, n, kernel="pair", split=[1, 2, 3, 0, 7, n - 13])
        b, _ = gpu_run(wl, n, kernel="stream")
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        assert_close(a, oracle_run(wl, n), "f64", f"pair {wl.name}")
    wl = workloads.make(3, nx=392, ny=250, steps=300)
    got, _ = gpu_run(wl, 300, dtype="f32", kernel="pair")
    assert_close(got, oracle_run(wl, 300), "f32", "pair cfg3 f32")


def test_pair_rectangular_mesh():
    wl = workloads.random_problem(6, 328, 150, batch=2, dy_ratio=0.6)
    got, _ = gpu_run(wl, 30, kernel="pair")
    assert_close(got, oracle_run(wl, 30), "f64", "pair dx != dy")


# ---------------------------------------------------------------------------------------------
# GG_KERNEL_QUAD: four steps per launch (two register-chained pair marches linked by a ring)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,nx", [("f64", 488), ("f32", 976)])
def test_quad_every_variant_and_chunking(dtype, nx):
    # three tile columns (fp64: 236 cells each, fp32: 472), the last one ragged
    wl = workloads.random_problem(45, nx, 150, batch=2)
    ref = {n: oracle_run(wl, n) for n in (4, 11)}
    base = {n: gpu_run(wl, n, dtype=dtype, kernel="stream")[0] for n in (4, 11)}
    for v in range(binding.gg_num_quad_variants()):
        for ipc, n in ((1, 4), (4, 11), (16, 4)):
            got, used = gpu_run(wl, n, dtype=dtype, kernel="quad",
                                options=[(binding.GG_OPT_QUAD_VARIANT, v), (binding.GG_OPT_ITEMS_PER_WARP, ipc)])
            assert used == "quad"
            assert_close(got, ref[n], dtype, f"quad {dtype} variant {v} items/CTA {ipc}")
            for x, y in zip(got, base[n]):
                assert np.array_equal(x, y), f"quad {dtype} variant {v}: not bit-identical"


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_quad_shapes_dtypes_and_boundaries(dtype):
    for nx, ny, batch in ((4, 2, 1), (8, 3, 2), (60, 17, 1), (236, 64, 1), (240, 40, 3), (472, 9, 1),
                          (1000, 37, 1), (2056, 70, 1)):
        wl = workloads.random_problem(400 + nx, nx, ny, batch=batch)
        for n in (4, 7, 8):
            got, used = gpu_run(wl, n, dtype=dtype, kernel="quad")
            assert used == "quad"
            assert_close(got, oracle_run(wl, n), dtype, f"quad {dtype} {nx}x{ny}x{batch} n={n}")


def test_quad_configs_long_runs_bit_identical_to_single_step():
    for wl, n in ((workloads.make(2, nx=520, ny=300, steps=200), 200),
                  (workloads.make(3, nx=392, ny=250, steps=300), 303),
                  (workloads.make(4, nx=264, ny=90, batch=5, steps=60), 60)):
        a, _ = gpu_run(wl, n, kernel="quad", split=[1, 2, 3, 0, 7, n - 13])
        b, _ = gpu_run(wl, n, kernel="stream")
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        assert_close(a, oracle_run(wl, n), "f64", f"quad {wl.name}")
    wl = workloads.make(3, nx=392, ny=250, steps=300)
    got, _ = gpu_run(wl, 300, dtype="f32", kernel="quad")
    assert_close(got, oracle_run(wl, 300), "f32", "quad cfg3 f32")
    wl = workloads.random_problem(7, 328, 150, batch=2, dy_ratio=0.6)
    got, _ = gpu_run(wl, 32, kernel="quad")
    assert_close(got, oracle_run(wl, 32), "f64", "quad dx != dy")


# ---------------------------------------------------------------------------------------------
# GG_KERNEL_RESIDENT: all n steps in one cooperative launch, state in shared memory
# ---------------------------------------------------------------------------------------------
# impl 0: one thread-block cluster per simulation where it fits (gg_cluster.cuh: distributed shared
# memory, every cell of a slab in parallel); impl 1: row slabs over the whole GPU (gg_resident.cuh)
@pytest.mark.parametrize("impl", [0, 1])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_resident_shapes_batches_and_ragged_slabs(dtype, impl):
    for nx, ny, batch in ((4, 2, 1), (8, 3, 2), (60, 17, 3), (64, 64, 1), (124, 41, 3), (200, 297, 1),
                          (512, 150, 1), (328, 150, 2), (64, 5, 40), (128, 128, 20)):
        if dtype == "f64" and nx > 512:
            continue
        if impl == 1 and batch > 5:
            continue                      # more slabs than SMs: only the cluster kernel takes these
        wl = workloads.random_problem(500 + nx, nx, ny, batch=batch)
        for n in (1, 2, 9):
            got, used = gpu_run(wl, n, dtype=dtype, kernel="resident", options=[(binding.GG_OPT_RESIDENT_IMPL, impl)])
            assert used == "resident"
            assert_close(got, oracle_run(wl, n), dtype, f"resident impl {impl} {dtype} {nx}x{ny}x{batch} n={n}")


@pytest.mark.parametrize("impl", [0, 1])
def test_resident_long_runs_bit_identical_to_single_step(impl):
    for wl, n in ((workloads.make(0), 200), (workloads.make(1, nx=256, ny=512, steps=400), 401),
                  (workloads.make(4, nx=264, ny=90, batch=5, steps=60), 60),
                  (workloads.random_problem(8, 328, 150, batch=2, dy_ratio=0.6), 33)):
        a, _ = gpu_run(wl, n, kernel="resident", split=[1, 2, 0, 7, n - 10], options=[(binding.GG_OPT_RESIDENT_IMPL, impl)])
        b, _ = gpu_run(wl, n, kernel="stream")
        for x, y in zip(a, b):
            assert np.array_equal(x, y)
        assert_close(a, oracle_run(wl, n), "f64", f"resident impl {impl} {wl.name}")


def test_resident_kernel_names():
    with binding.from_workload(workloads.make(0)) as sim:
        assert sim.kernel == "resident" and sim.kernel_name == "gg_step_cluster<double,1>"
        sim.set_option(binding.GG_OPT_RESIDENT_IMPL, 1)
        assert sim.kernel_name == "gg_step_resident<double>"


def test_two_live_contexts_interleaved():
    """Two contexts of different shapes alive at once, stepped alternately, on the kernels whose
    dynamic shared-memory size depends on the shape (resident, cluster, pair): per-function
    attributes must not leak from one context into the other."""
    wa, wb = workloads.random_problem(71, 512, 96), workloads.random_problem(72, 64, 48)
    for kernel, opts in (("resident", [(binding.GG_OPT_RESIDENT_IMPL, 1)]), ("resident", []), ("pair", [])):
        with binding.from_workload(wa, dtype="f32") as sa, binding.from_workload(wb, dtype="f32") as sb:
            for sim in (sa, sb):
                sim.set_option(binding.GG_OPT_KERNEL, KERNELS[kernel])
                for o, v in opts:
                    sim.set_option(o, v)
            for _ in range(3):
                sa.step(4, wa.dt)
                sb.step(4, wb.dt)
            ga, gb = sa.get_state_numpy(), sb.get_state_numpy()
        assert_close(ga, oracle_run(wa, 12), "f32", f"two contexts {kernel} (a)")
        assert_close(gb, oracle_run(wb, 12), "f32", f"two contexts {kernel} (b)")


def test_resident_refuses_grids_that_do_not_fit():
    wl = workloads.make(2, nx=1024, ny=64, steps=1)          # 8 KB rows: more than 256 lanes
    with binding.from_workload(wl) as sim:
        assert sim.kernel != "resident"
        with pytest.raises(binding.GGError) as e:
            sim.set_option(binding.GG_OPT_KERNEL, binding.GG_KERNEL_RESIDENT)
        assert e.value.code == binding.GG_ERR_UNSUPPORTED
    wl = workloads.make(2, nx=64, ny=16384, steps=1)         # more 64-row slabs than SMs
    with binding.from_workload(wl) as sim:
        assert sim.kernel != "resident"


def test_user_stream_every_auto_path():
    """The library enqueues on the stream given to gg_bind: run the resident, quad (whose odd step
    counts end with a pair and a single-step launch) and generic paths on a non-default stream
    while the default stream is kept busy."""
    import torch
    stream = torch.cuda.Stream()
    busy = torch.empty(64 << 20, device="cuda")
    for wl, n, want, dtype in ((workloads.make(0), 40, "resident", "f64"),
                               (workloads.make(1, nx=512, ny=160, steps=1), 24, "quad", "f64"),
                               (workloads.make(3, nx=2048, ny=800, steps=1), 11, "quad", "f32"),
                               (workloads.make(3, nx=1200, ny=400, steps=1), 12, "quad", "f32"),
                               (workloads.random_problem(3, 41, 23), 9, "generic", "f64")):
        for _ in range(4):
            busy.add_(1.0)                       # unrelated work on the default stream
        with binding.from_workload(wl, dtype=dtype, stream=stream) as sim:
            assert sim.kernel == want
            sim.step(n, wl.dt)
            got = sim.get_state_numpy()
        assert_close(got, oracle_run(wl, n), dtype, f"user stream {want}")


def test_split_calls_equal_one_call():
    wl = workloads.make(1, nx=128, ny=96)
    a, _ = gpu_run(wl, 37)
    b, _ = gpu_run(wl, 37, split=[1, 0, 3, 20, 13])
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert_close(a, oracle_run(wl, 37), "f64", "split")


def test_zero_steps_and_roundtrip():
    wl = workloads.random_problem(3, 32, 16, batch=3)
    with binding.from_workload(wl) as sim:
        sim.step(0, wl.dt)
        U, V, W = sim.get_state_numpy()
        assert sim.launches == 0
    assert np.array_equal(U, wl.U) and np.array_equal(V, wl.V) and np.array_equal(W, wl.W)


def test_host_buffer_entry_points():
    wl = workloads.random_problem(11, 96, 40)
    with binding.Simulation(wl.nx, wl.ny, wl.h, wl.r, wl.d, wl.alpha, wl.c_r) as sim:
        sim.set_tensor_host(wl.a, wl.b, wl.c)
        sim.set_state_host(wl.U, wl.V, wl.W)
        sim.step(6, wl.dt)
        out = [np.empty_like(wl.U) for _ in range(3)]
        sim.get_state_host(*out)
        assert sim.last_step_ms() >= 0.0
    assert_close(out, oracle_run(wl, 6), "f64", "host entry points")


def test_errors_on_device():
    wl = workloads.random_problem(1, 16, 8)
    with binding.from_workload(wl) as sim:
        for bad in (0.0, -1.0, float("nan"), float("inf")):
            with pytest.raises(binding.GGError) as e:
                sim.step(1, bad)
            assert e.value.code == binding.GG_ERR_ARG
        with pytest.raises(binding.GGError):
            sim.step(-1, wl.dt)
    with binding.Simulation(16, 8, wl.h, 1, 1, 1, 1) as sim:
        with pytest.raises(binding.GGError) as e:
            sim.step(1, wl.dt)  # no tensor / state yet
        assert e.value.code == binding.GG_ERR_STATE


# ---------------------------------------------------------------------------------------------
# physics invariants on the GPU result itself (hold at any size)
# ---------------------------------------------------------------------------------------------
def test_equilibria_and_uniform_data_on_gpu():
    wl = workloads.random_problem(8, 128, 64)
    one, zero = np.ones_like(wl.U), np.zeros_like(wl.U)
    for (u, v, w) in [(one, zero, zero), (zero, one, one), (zero, zero, zero)]:
        wl.U, wl.V, wl.W = u, v, w
        got, _ = gpu_run(wl, 20)
        assert np.array_equal(got[0], u) and np.array_equal(got[1], v) and np.array_equal(got[2], w)


def test_mass_conservation_on_gpu():
    wl = workloads.random_problem(9, 256, 128)
    wl.c_r[:] = 0.0
    wl.r[:] = 0.0
    got, _ = gpu_run(wl, 200)
    assert abs(got[2].sum() - wl.W.sum()) <= 1e-12 * wl.W.sum()
    assert abs(got[1].sum() - wl.V.sum()) <= 1e-12 * wl.V.sum()


def test_fp32_packed_arithmetic_keeps_denormals():
    """The fp32 four-step kernel computes on packed pairs of cells (FADD2 / FMUL2 / FFMA2); the
    single-step kernel is scalar.  Far from the tumour the acid field decays into the denormal
    range: the packed instructions must round those exactly as the scalar ones (no flush to zero)."""
    wl = workloads.random_problem(77, 944, 64)
    wl.W *= 1e-39                       # denormal in fp32
    wl.V *= 1e-38
    wl.U[:] = 1.0 - 1e-7 * wl.U
    a, _ = gpu_run(wl, 12, dtype="f32", kernel="quad")
    b, _ = gpu_run(wl, 12, dtype="f32", kernel="stream")
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    assert np.any((np.abs(a[2]) > 0) & (np.abs(a[2]) < 1.1754944e-38))   # denormals really occur
