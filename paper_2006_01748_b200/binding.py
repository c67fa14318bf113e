"""Thin ctypes binding of libgg.so (include/gg.h): argument marshalling only.

Every step of the method runs inside the library's CUDA kernels; this module converts Python
arguments to C ones, lets PyTorch own device memory and the stream, and raises `GGError` on a
non-zero status.  There is no CPU fallback: if libgg.so is missing and cannot be built, or no
CUDA device is present, the calls fail loudly.

Function names mirror the C ABI (`gg_create`, `gg_set_tensor`, `gg_set_state`, `gg_step`,
`gg_get_state`, ...).  `Simulation` is a small convenience holder that owns the torch workspace
tensor and forwards to those functions.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

GG_F64, GG_F32 = 0, 1
GG_OK, GG_ERR_ARG, GG_ERR_STATE, GG_ERR_CUDA, GG_ERR_UNSUPPORTED = 0, 1, 2, 3, 4
GG_KERNEL_AUTO, GG_KERNEL_GENERIC, GG_KERNEL_STREAM, GG_KERNEL_STREAM2, GG_KERNEL_RESIDENT, \
    GG_KERNEL_PAIR, GG_KERNEL_QUAD = range(7)
GG_OPT_KERNEL, GG_OPT_GRAPH, GG_OPT_GRAPH_CHUNK, GG_OPT_STREAM_VARIANT, GG_OPT_ITEMS_PER_WARP, \
    GG_OPT_STREAM_WARPS, GG_OPT_STREAM2_VARIANT, GG_OPT_PAIR_VARIANT, GG_OPT_QUAD_VARIANT, \
    GG_OPT_RESIDENT_IMPL, GG_OPT_CLUSTER_CTAS = range(11)

KERNEL_NAMES = {GG_KERNEL_AUTO: "auto", GG_KERNEL_GENERIC: "generic", GG_KERNEL_STREAM: "stream",
                GG_KERNEL_STREAM2: "stream2", GG_KERNEL_RESIDENT: "resident", GG_KERNEL_PAIR: "pair", GG_KERNEL_QUAD: "quad"}

_vp = ctypes.c_void_p
_dp = ctypes.POINTER(ctypes.c_double)

# name -> (restype, argtypes); the CPU test tier checks every name against include/gg.h
SIGNATURES = {
    "gg_create": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                 ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                 ctypes.c_double, ctypes.c_int]),
    "gg_create_batch": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int,
                                       ctypes.c_int, ctypes.c_double, _dp, _dp, _dp, _dp,
                                       ctypes.c_int]),
    "gg_create_xy": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_double, ctypes.c_double, _dp, _dp, _dp, _dp,
                                    ctypes.c_int]),
    "gg_workspace_bytes": (ctypes.c_size_t, [_vp]),
    "gg_bind": (ctypes.c_int, [_vp, _vp, ctypes.c_size_t, _vp]),
    "gg_set_tensor": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_set_state": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_step": (ctypes.c_int, [_vp, ctypes.c_longlong, ctypes.c_double]),
    "gg_step_adaptive": (ctypes.c_int, [_vp, ctypes.c_longlong, ctypes.c_double, ctypes.c_longlong]),
    "gg_get_clock": (ctypes.c_int, [_vp, _dp, _dp, ctypes.POINTER(ctypes.c_longlong)]),
    "gg_get_state": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_set_tensor_host": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_set_state_host": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_get_state_host": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "gg_diagnostics": (ctypes.c_int, [_vp, ctypes.c_double, _dp]),
    "gg_diagnostics_noalloc": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_double, _vp, _vp]),
    "gg_noalloc_last_error": (ctypes.c_char_p, []),
    "gg_max_stable_dt": (ctypes.c_int, [_vp, ctypes.c_double, _dp, _dp]),
    "gg_front": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                ctypes.POINTER(ctypes.c_int)]),
    "gg_set_option": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_longlong]),
    "gg_kernel_used": (ctypes.c_int, [_vp]),
    "gg_kernel_name": (ctypes.c_char_p, [_vp]),
    "gg_launches": (ctypes.c_longlong, [_vp]),
    "gg_graph_captures": (ctypes.c_longlong, [_vp]),
    "gg_last_step_ms": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_float)]),
    "gg_destroy": (ctypes.c_int, [_vp]),
    "gg_last_error": (ctypes.c_char_p, [_vp]),
    "gg_version": (ctypes.c_char_p, []),
}
# tuning entry points of the non-installed csrc/gg_tuning.h (tests force every build through parity)
TUNING_SIGNATURES = {
    "gg_num_stream_variants": (ctypes.c_int, []),
    "gg_num_stream2_variants": (ctypes.c_int, []),
    "gg_num_pair_variants": (ctypes.c_int, []),
    "gg_num_quad_variants": (ctypes.c_int, []),
}

_lib = None


class GGError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libgg error {code}: {msg}")
        self.code = code


def load() -> ctypes.CDLL:
    """dlopen libgg.so (building it in-tree with nvcc first if it is missing or stale)."""
    global _lib
    if _lib is None:
        path = _build.build() if os.path.exists(_build.NVCC) else _build.LIB
        if not os.path.exists(path):
            raise RuntimeError("libgg.so is missing and nvcc is not available to build it; "
                               "there is no CPU fallback")
        lib = ctypes.CDLL(path)
        for name, (res, args) in {**SIGNATURES, **TUNING_SIGNATURES}.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(ctx, rc: int):
    if rc != GG_OK:
        raise GGError(rc, (load().gg_last_error(ctx) or b"").decode())


def _darr(x, n):
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(x, dtype=np.float64), (n,)))
    return a, a.ctypes.data_as(_dp)


# ---- functions named after the C ABI ---------------------------------------------------------
def gg_create(nx, ny, h, r, d, alpha, c, dtype=GG_F64):
    ctx = _vp()
    _check(None, load().gg_create(ctypes.byref(ctx), nx, ny, h, r, d, alpha, c, dtype))
    return ctx


def gg_create_batch(nbatch, nx, ny, h, r, d, alpha, c, dtype=GG_F64):
    ctx = _vp()
    keep = [_darr(v, nbatch) for v in (r, d, alpha, c)]
    _check(None, load().gg_create_batch(ctypes.byref(ctx), nbatch, nx, ny, h,
                                        *[k[1] for k in keep], dtype))
    return ctx


def gg_create_xy(nbatch, nx, ny, dx, dy, r, d, alpha, c, dtype=GG_F64):
    ctx = _vp()
    keep = [_darr(v, nbatch) for v in (r, d, alpha, c)]
    _check(None, load().gg_create_xy(ctypes.byref(ctx), nbatch, nx, ny, dx, dy,
                                     *[k[1] for k in keep], dtype))
    return ctx


def gg_workspace_bytes(ctx) -> int:
    return int(load().gg_workspace_bytes(ctx))


def gg_bind(ctx, workspace_ptr: int, nbytes: int, stream_ptr: int = 0):
    _check(ctx, load().gg_bind(ctx, workspace_ptr, nbytes, stream_ptr))


def gg_set_tensor(ctx, a_ptr, b_ptr, c_ptr):
    _check(ctx, load().gg_set_tensor(ctx, a_ptr, b_ptr, c_ptr))


def gg_set_state(ctx, U_ptr, V_ptr, W_ptr):
    _check(ctx, load().gg_set_state(ctx, U_ptr, V_ptr, W_ptr))


def gg_step(ctx, n: int, dt: float):
    _check(ctx, load().gg_step(ctx, int(n), float(dt)))


def gg_step_adaptive(ctx, n: int, safety: float, every_k: int):
    _check(ctx, load().gg_step_adaptive(ctx, int(n), float(safety), int(every_k)))


def gg_get_clock(ctx):
    """(time, dt of the most recent step, steps) of the device-side clock."""
    t, dt, n = ctypes.c_double(0.0), ctypes.c_double(0.0), ctypes.c_longlong(0)
    _check(ctx, load().gg_get_clock(ctx, ctypes.byref(t), ctypes.byref(dt), ctypes.byref(n)))
    return float(t.value), float(dt.value), int(n.value)


def gg_get_state(ctx, U_ptr, V_ptr, W_ptr):
    _check(ctx, load().gg_get_state(ctx, U_ptr, V_ptr, W_ptr))


def gg_set_tensor_host(ctx, a_ptr, b_ptr, c_ptr):
    _check(ctx, load().gg_set_tensor_host(ctx, a_ptr, b_ptr, c_ptr))


def gg_set_state_host(ctx, U_ptr, V_ptr, W_ptr):
    _check(ctx, load().gg_set_state_host(ctx, U_ptr, V_ptr, W_ptr))


def gg_get_state_host(ctx, U_ptr, V_ptr, W_ptr):
    _check(ctx, load().gg_get_state_host(ctx, U_ptr, V_ptr, W_ptr))


GG_DIAG_NAMES = ("sum_U", "sum_V", "sum_W", "gap_cells", "tumour_cells", "min_W", "max_U", "max_W",
                 "nonfinite_cells")
GG_DIAG_COUNT = len(GG_DIAG_NAMES)


def gg_diagnostics(ctx, eps: float, nbatch: int) -> np.ndarray:
    """[nbatch][GG_DIAG_COUNT] doubles, slot order GG_DIAG_NAMES."""
    out = np.empty((nbatch, GG_DIAG_COUNT), dtype=np.float64)
    _check(ctx, load().gg_diagnostics(ctx, float(eps), out.ctypes.data_as(_dp)))
    return out


GG_NOALLOC_MAX_BATCH = 64


def gg_noalloc_last_error() -> str:
    return (load().gg_noalloc_last_error() or b"").decode()


def gg_diagnostics_noalloc(U_ptr, V_ptr, W_ptr, nbatch: int, nx: int, ny: int, dtype: int, eps: float,
                           out_ptr, stream_ptr: int = 0):
    """The context-free, allocation-free diagnostics call for callers that cannot allocate device
    memory (gg.h): U, V, W and `out` ([nbatch][GG_DIAG_COUNT] doubles) are DEVICE pointers the
    caller owns; the result is in `out` once `stream_ptr` has reached this point.  Enqueues only."""
    rc = load().gg_diagnostics_noalloc(U_ptr, V_ptr, W_ptr, int(nbatch), int(nx), int(ny), int(dtype),
                                       float(eps), out_ptr, stream_ptr)
    if rc != GG_OK:
        raise GGError(rc, gg_noalloc_last_error())


def gg_front(ctx, field: int, axis: int, index: int, level: float, nbatch: int) -> np.ndarray:
    """[nbatch][2] ints: first and last cell index along the line with field >= level, or -1."""
    out = np.empty((nbatch, 2), dtype=np.int32)
    _check(ctx, load().gg_front(ctx, int(field), int(axis), int(index), float(level),
                                out.ctypes.data_as(ctypes.POINTER(ctypes.c_int))))
    return out


def gg_max_stable_dt(ctx, safety: float):
    """(dt, lambda_max)."""
    dt, lam = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(ctx, load().gg_max_stable_dt(ctx, float(safety), ctypes.byref(dt), ctypes.byref(lam)))
    return float(dt.value), float(lam.value)


def gg_set_option(ctx, option: int, value: int):
    _check(ctx, load().gg_set_option(ctx, option, int(value)))


def gg_kernel_used(ctx) -> int:
    return int(load().gg_kernel_used(ctx))


def gg_kernel_name(ctx) -> str:
    return (load().gg_kernel_name(ctx) or b"").decode()


def gg_launches(ctx) -> int:
    return int(load().gg_launches(ctx))


def gg_graph_captures(ctx) -> int:
    return int(load().gg_graph_captures(ctx))


def gg_last_step_ms(ctx) -> float:
    ms = ctypes.c_float(-1.0)
    _check(ctx, load().gg_last_step_ms(ctx, ctypes.byref(ms)))
    return float(ms.value)


def gg_destroy(ctx):
    _check(None, load().gg_destroy(ctx))


def gg_last_error(ctx=None) -> str:
    return (load().gg_last_error(ctx) or b"").decode()


def gg_version() -> str:
    return load().gg_version().decode()


def gg_num_stream_variants() -> int:
    return int(load().gg_num_stream_variants())


def gg_num_stream2_variants() -> int:
    return int(load().gg_num_stream2_variants())


def gg_num_pair_variants() -> int:
    return int(load().gg_num_pair_variants())


def gg_num_quad_variants() -> int:
    return int(load().gg_num_quad_variants())


# ---- convenience holder (torch owns device memory and the stream) ------------------------------
class Simulation:
    """One context + its torch workspace.  Marshalling only; all arithmetic is in libgg.so.

    r, d, alpha, c are scalars or length-`batch` sequences.  `dtype` is "f64" or "f32".
    `h` is the mesh size dx; pass `dy=` for a non-square mesh.
    """

    def __init__(self, nx, ny, h, r, d, alpha, c, dtype="f64", batch=1, device="cuda:0",
                 stream=None, dy=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2006_01748_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.nx, self.ny, self.batch = int(nx), int(ny), int(batch)
        self.dtype = {"f64": GG_F64, "f32": GG_F32}[dtype]
        self.tdtype = torch.float64 if self.dtype == GG_F64 else torch.float32
        self.npdtype = np.float64 if self.dtype == GG_F64 else np.float32
        torch.cuda.set_device(self.device)
        # h is dx; dy defaults to it (square mesh)
        self.ctx = gg_create_xy(self.batch, self.nx, self.ny, float(h),
                                float(h if dy is None else dy), r, d, alpha, c, self.dtype)
        nbytes = gg_workspace_bytes(self.ctx)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self.stream = stream
        sptr = 0 if stream is None else int(stream.cuda_stream)
        gg_bind(self.ctx, self._ws_ptr, nbytes, sptr)

    # device tensors ---------------------------------------------------------------------------
    def _dev(self, x, shape):
        t = self.torch.as_tensor(x)
        t = t.to(device=self.device, dtype=self.tdtype).contiguous()
        if tuple(t.shape) != shape:
            t = t.reshape(shape)
        return t

    def set_tensor(self, a, b, c):
        sh = (self.ny, self.nx)
        ta, tb, tc = (self._dev(x, sh) for x in (a, b, c))
        self._after_current_stream()
        gg_set_tensor(self.ctx, ta.data_ptr(), tb.data_ptr(), tc.data_ptr())
        self._sync()  # temporaries may be freed after return

    def set_state(self, U, V, W):
        sh = (self.batch, self.ny, self.nx)
        tU, tV, tW = (self._dev(x, sh) for x in (U, V, W))
        self._after_current_stream()
        gg_set_state(self.ctx, tU.data_ptr(), tV.data_ptr(), tW.data_ptr())
        self._sync()

    def step(self, n, dt):
        gg_step(self.ctx, n, dt)

    def step_adaptive(self, n, safety=0.2, every_k=1):
        gg_step_adaptive(self.ctx, n, safety, every_k)

    def clock(self):
        return gg_get_clock(self.ctx)

    @property
    def graph_captures(self) -> int:
        return gg_graph_captures(self.ctx)

    def get_state(self):
        """Current (U, V, W) as device tensors [batch][ny][nx]."""
        sh = (self.batch, self.ny, self.nx)
        out = [self.torch.empty(sh, dtype=self.tdtype, device=self.device) for _ in range(3)]
        gg_get_state(self.ctx, *(t.data_ptr() for t in out))
        self._sync()
        return tuple(out)

    def get_state_numpy(self):
        return tuple(t.cpu().numpy() for t in self.get_state())

    # host buffers (numpy arrays of the context dtype, C-contiguous) ----------------------------
    def set_tensor_host(self, a, b, c):
        arrs = [np.ascontiguousarray(x, dtype=self.npdtype) for x in (a, b, c)]
        gg_set_tensor_host(self.ctx, *(x.ctypes.data for x in arrs))

    def set_state_host(self, U, V, W):
        arrs = [np.ascontiguousarray(x, dtype=self.npdtype) for x in (U, V, W)]
        gg_set_state_host(self.ctx, *(x.ctypes.data for x in arrs))

    def get_state_host(self, U, V, W):
        for x in (U, V, W):
            assert x.dtype == self.npdtype and x.flags["C_CONTIGUOUS"]
        gg_get_state_host(self.ctx, U.ctypes.data, V.ctypes.data, W.ctypes.data)

    def diagnostics(self, eps=1e-2):
        return gg_diagnostics(self.ctx, eps, self.batch)

    def front(self, field, axis, index, level=0.5):
        return gg_front(self.ctx, {"U": 0, "V": 1, "W": 2}.get(field, field), axis, index, level, self.batch)

    def max_stable_dt(self, safety=0.2):
        return gg_max_stable_dt(self.ctx, safety)

    # options / introspection ------------------------------------------------------------------
    def set_option(self, option, value):
        gg_set_option(self.ctx, option, value)

    @property
    def kernel(self) -> str:
        return KERNEL_NAMES.get(gg_kernel_used(self.ctx), "?")

    @property
    def kernel_name(self) -> str:
        return gg_kernel_name(self.ctx)

    @property
    def launches(self) -> int:
        return gg_launches(self.ctx)

    def last_step_ms(self) -> float:
        return gg_last_step_ms(self.ctx)

    def _after_current_stream(self):
        """libgg enqueues on the bound stream; tensors staged by torch live on torch's current
        stream (inputs must be ready there): order the bound stream after it, also when the
        bound stream is the legacy default stream -- torch side streams are non-blocking and not
        implicitly ordered with it (stream plumbing only)."""
        cur = self.torch.cuda.current_stream(self.device)
        if self.stream is not None:
            self.stream.wait_stream(cur)
        elif int(cur.cuda_stream) != 0:
            cur.synchronize()

    def _sync(self):
        if self.stream is None:
            self.torch.cuda.synchronize(self.device)
        else:
            self.stream.synchronize()

    def close(self):
        if getattr(self, "ctx", None) is not None:
            gg_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def from_workload(wl, dtype="f64", **kw) -> Simulation:
    """Build a Simulation from a `workloads.Workload` and load its tensor and initial state."""
    sim = Simulation(wl.nx, wl.ny, wl.h, wl.r, wl.d, wl.alpha, wl.c_r, dtype=dtype, batch=wl.batch,
                     dy=wl.dy, **kw)
    sim.set_tensor(wl.a, wl.b, wl.c)
    sim.set_state(wl.U, wl.V, wl.W)
    return sim
