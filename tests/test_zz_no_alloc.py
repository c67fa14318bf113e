"""GPU test (-m gpu) of gg_diagnostics_noalloc, the one call of the library that takes no context
and no workspace and allocates nothing itself.

Why the call exists: every other entry point works on memory the caller allocated for it
(gg_workspace_bytes / gg_bind).  Some callers have none to give -- a probe that another program's
time loop calls with just the device pointers of its fields, a plug-in inside an application whose
pool already holds the whole GPU, a hook that must not trigger the device-wide synchronisation a
cudaMalloc implies.  For them the partial sums of the reduction sit in a fixed 1.3 MiB array built
into libgg.so's device image (at most GG_NOALLOC_MAX_BATCH = 64 simulations per call).

What is checked: on the same device-resident fields the call returns what the existing
gg_diagnostics path returns -- counts, minima and maxima exactly, the three sums to the 1e-12 the
reduction tests use (the two paths add the same numbers in a different order) -- on TWO calls in a
row whose shapes, batch sizes and contents differ, so that anything the first call left behind in
the shared array (stale partials of a larger grid, arrival counters) would corrupt the second.  A
third call repeats the first and must reproduce it bit for bit.  Oversized batches and bad arguments
are refused with a message.

This file is named to be collected last: with `pytest -x` a failure here cannot hide the parity
tests.  It needs nothing the other tests set up and leaves nothing behind, so it passes alone in a
fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2006_01748_b200 import binding, workloads

pytestmark = pytest.mark.gpu


def check_diag(got, ref):
    """tests/test_gpu_reductions.py's tolerance: sums 1e-12, everything else exact."""
    np.testing.assert_allclose(got[:3], ref[:3], rtol=1e-12, atol=1e-12)
    assert list(got[3:]) == list(ref[3:])


def both_paths(wl, dtype, steps, eps):
    """(existing path, new entry point) on the very same device state after `steps` steps."""
    import torch
    with binding.from_workload(wl, dtype=dtype) as sim:
        if steps:
            sim.step(steps, wl.dt)
        ref = sim.diagnostics(eps)                       # gg_diagnostics: context + workspace
        U, V, W = sim.get_state()                        # caller-owned device tensors
        out = torch.full((wl.batch, binding.GG_DIAG_COUNT), float("nan"), dtype=torch.float64, device=U.device)
        torch.cuda.synchronize()
        binding.gg_diagnostics_noalloc(U.data_ptr(), V.data_ptr(), W.data_ptr(), wl.batch, wl.nx, wl.ny,
                                       sim.dtype, eps, out.data_ptr(), 0)
        torch.cuda.synchronize()
        return ref, out.cpu().numpy()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_noalloc_matches_the_workspace_path_on_two_calls_in_a_row(dtype):
    # call 1: many segments per simulation (296 partial blocks, ragged tail), b != 0 undershoot
    big = workloads.make(4, nx=1032, ny=515, batch=3, steps=12)
    # call 2: fewer, shorter segments and MORE simulations than call 1 used -- reads nothing stale
    small = workloads.make(4, nx=263, ny=190, batch=7, steps=40)   # odd width: unaligned planes, scalar loads
    ref1, got1 = both_paths(big, dtype, big.steps, 0.3)
    ref2, got2 = both_paths(small, dtype, small.steps, 1e-2)
    for s in range(big.batch):
        check_diag(got1[s], ref1[s])
    for s in range(small.batch):
        check_diag(got2[s], ref2[s])
    assert not np.array_equal(got2[0], got2[-1])          # different d per simulation: really per-simulation
    assert np.all(ref1[:, 2] != 0) and np.all(ref1[:, 4] > 0)   # stepped fields: acid present, tumour cells counted
    # call 3 = call 1 again, after call 2 overwrote the shared scratch: bit-identical (fixed order)
    _, again = both_paths(big, dtype, big.steps, 0.3)
    assert np.array_equal(again, got1)


def test_noalloc_full_batch_and_limit():
    import torch
    nb = binding.GG_NOALLOC_MAX_BATCH
    wl = workloads.make(4, nx=64, ny=48, batch=nb, steps=0)
    ref, got = both_paths(wl, "f64", 0, 0.05)
    for s in range(nb):
        check_diag(got[s], ref[s])
    # one simulation more than the built-in scratch holds: refused, with a message, nothing launched
    z = torch.zeros((nb + 1, 4, 4), dtype=torch.float64, device="cuda:0")
    out = torch.zeros((nb + 1, binding.GG_DIAG_COUNT), dtype=torch.float64, device="cuda:0")
    with pytest.raises(binding.GGError) as e:
        binding.gg_diagnostics_noalloc(z.data_ptr(), z.data_ptr(), z.data_ptr(), nb + 1, 4, 4, binding.GG_F64, 0.1,
                                       out.data_ptr(), 0)
    assert e.value.code == binding.GG_ERR_ARG and "GG_NOALLOC_MAX_BATCH" in str(e.value)
    for kw in (dict(nbatch=0), dict(nx=0), dict(eps=-1.0), dict(eps=float("nan")), dict(dtype=5), dict(out=0)):
        a = dict(nbatch=1, nx=4, ny=4, dtype=binding.GG_F64, eps=0.1, out=out.data_ptr())
        a.update(kw)
        with pytest.raises(binding.GGError) as e:
            binding.gg_diagnostics_noalloc(z.data_ptr(), z.data_ptr(), z.data_ptr(), a["nbatch"], a["nx"], a["ny"],
                                           a["dtype"], a["eps"], a["out"], 0)
        assert e.value.code in (binding.GG_ERR_ARG, binding.GG_ERR_UNSUPPORTED) and str(e.value)


def test_noalloc_on_a_side_stream_with_known_values():
    """Values a reader can check by hand, on a non-default stream: U = 1, V = 0 except one cell at
    0.75, W = -2 in one cell, +3 in another, one NaN in U of the second simulation."""
    import torch
    dev = torch.device("cuda:0")
    nb, ny, nx = 2, 37, 41
    U = torch.ones((nb, ny, nx), dtype=torch.float32, device=dev)
    V = torch.zeros_like(U)
    W = torch.zeros_like(U)
    V[0, 5, 7] = 0.75
    W[0, 36, 40] = -2.0
    W[1, 0, 0] = 3.0
    U[1, 20, 20] = float("nan")
    out = torch.empty((nb, binding.GG_DIAG_COUNT), dtype=torch.float64, device=dev)
    side = torch.cuda.Stream(device=dev)
    side.wait_stream(torch.cuda.current_stream(dev))
    binding.gg_diagnostics_noalloc(U.data_ptr(), V.data_ptr(), W.data_ptr(), nb, nx, ny, binding.GG_F32, 0.5,
                                   out.data_ptr(), int(side.cuda_stream))
    side.synchronize()
    got = out.cpu().numpy()
    n = nx * ny
    assert list(got[0]) == [n, 0.75, -2.0, 0.0, 1.0, -2.0, 1.0, 0.0, 0.0]
    assert np.isnan(got[1][0]) and list(got[1][1:]) == [0.0, 3.0, 0.0, 0.0, 0.0, 1.0, 3.0, 1.0]
