"""ctypes binding of include/gg3.h (the three-dimensional extension): the same names as the C ABI,
argument marshalling only -- every step of the path runs in libgg.so.  No CPU fallback."""
from __future__ import annotations

import ctypes

import numpy as np

from . import binding as _b

_vp = ctypes.c_void_p
GG3_KERNEL_AUTO, GG3_KERNEL_GENERIC, GG3_KERNEL_TILED = range(3)
GG3_OPT_KERNEL, GG3_OPT_GRAPH, GG3_OPT_GRAPH_CHUNK = range(3)
KERNEL_NAMES = {GG3_KERNEL_GENERIC: "generic", GG3_KERNEL_TILED: "tiled"}

SIGNATURES = {
    "gg3_create": (ctypes.c_int, [ctypes.POINTER(_vp)] + [ctypes.c_int] * 3 + [ctypes.c_double] * 7 + [ctypes.c_int]),
    "gg3_workspace_bytes": (ctypes.c_size_t, [_vp]),
    "gg3_bind": (ctypes.c_int, [_vp, _vp, ctypes.c_size_t, _vp]),
    "gg3_set_tensor": (ctypes.c_int, [_vp] * 7),
    "gg3_set_tensor_host": (ctypes.c_int, [_vp] * 7),
    "gg3_set_state": (ctypes.c_int, [_vp] * 4),
    "gg3_set_state_host": (ctypes.c_int, [_vp] * 4),
    "gg3_step": (ctypes.c_int, [_vp, ctypes.c_longlong, ctypes.c_double]),
    "gg3_get_state": (ctypes.c_int, [_vp] * 4),
    "gg3_get_state_host": (ctypes.c_int, [_vp] * 4),
    "gg3_set_option": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_longlong]),
    "gg3_kernel_used": (ctypes.c_int, [_vp]),
    "gg3_launches": (ctypes.c_longlong, [_vp]),
    "gg3_graph_captures": (ctypes.c_longlong, [_vp]),
    "gg3_last_step_ms": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_float)]),
    "gg3_destroy": (ctypes.c_int, [_vp]),
    "gg3_last_error": (ctypes.c_char_p, [_vp]),
}
_ready = False


def load() -> ctypes.CDLL:
    global _ready
    lib = _b.load()
    if not _ready:
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _ready = True
    return lib


def _check(ctx, rc: int):
    if rc != _b.GG_OK:
        raise _b.GGError(rc, (load().gg3_last_error(ctx) or b"").decode())


# ---- functions named after the C ABI ---------------------------------------------------------
def gg3_create(nx, ny, nz, dx, dy, dz, r, d, alpha, c, dtype=_b.GG_F64):
    ctx = _vp()
    _check(None, load().gg3_create(ctypes.byref(ctx), nx, ny, nz, dx, dy, dz, r, d, alpha, c, dtype))
    return ctx


def gg3_workspace_bytes(ctx) -> int:
    return int(load().gg3_workspace_bytes(ctx))


def gg3_bind(ctx, ws_ptr, nbytes, stream_ptr=0):
    _check(ctx, load().gg3_bind(ctx, ws_ptr, nbytes, stream_ptr))


def gg3_set_tensor(ctx, *ptrs):
    _check(ctx, load().gg3_set_tensor(ctx, *ptrs))


def gg3_set_tensor_host(ctx, *ptrs):
    _check(ctx, load().gg3_set_tensor_host(ctx, *ptrs))


def gg3_set_state(ctx, U, V, W):
    _check(ctx, load().gg3_set_state(ctx, U, V, W))


def gg3_set_state_host(ctx, U, V, W):
    _check(ctx, load().gg3_set_state_host(ctx, U, V, W))


def gg3_step(ctx, n, dt):
    _check(ctx, load().gg3_step(ctx, int(n), float(dt)))


def gg3_get_state(ctx, U, V, W):
    _check(ctx, load().gg3_get_state(ctx, U, V, W))


def gg3_get_state_host(ctx, U, V, W):
    _check(ctx, load().gg3_get_state_host(ctx, U, V, W))


def gg3_set_option(ctx, option, value):
    _check(ctx, load().gg3_set_option(ctx, int(option), int(value)))


def gg3_kernel_used(ctx) -> int:
    return int(load().gg3_kernel_used(ctx))


def gg3_launches(ctx) -> int:
    return int(load().gg3_launches(ctx))


def gg3_graph_captures(ctx) -> int:
    return int(load().gg3_graph_captures(ctx))


def gg3_last_step_ms(ctx) -> float:
    ms = ctypes.c_float()
    _check(ctx, load().gg3_last_step_ms(ctx, ctypes.byref(ms)))
    return float(ms.value)


def gg3_destroy(ctx):
    load().gg3_destroy(ctx)


def gg3_last_error(ctx) -> str:
    return (load().gg3_last_error(ctx) or b"").decode()


# ---- convenience holder (torch owns device memory) ----------------------------------------------
class Simulation3:
    """One 3-D context + its torch workspace.  Marshalling only."""

    def __init__(self, nx, ny, nz, dx, dy, dz, r, d, alpha, c, dtype="f64", device="cuda:0"):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2006_01748_b200 needs a CUDA device; there is no CPU fallback")
        self.torch, self.device = torch, torch.device(device)
        self.shape = (int(nz), int(ny), int(nx))
        self.dtype = {"f64": _b.GG_F64, "f32": _b.GG_F32}[dtype]
        self.tdtype = torch.float64 if self.dtype == _b.GG_F64 else torch.float32
        torch.cuda.set_device(self.device)
        self.ctx = gg3_create(nx, ny, nz, float(dx), float(dy), float(dz), float(r), float(d), float(alpha), float(c), self.dtype)
        nbytes = gg3_workspace_bytes(self.ctx)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        gg3_bind(self.ctx, (self.workspace.data_ptr() + 255) // 256 * 256, nbytes, 0)

    def _dev(self, x):
        return self.torch.as_tensor(np.ascontiguousarray(x)).to(device=self.device, dtype=self.tdtype).reshape(self.shape).contiguous()

    def set_tensor(self, tensor):
        ts = [self._dev(t) for t in tensor]
        self.torch.cuda.current_stream(self.device).synchronize()
        gg3_set_tensor(self.ctx, *(t.data_ptr() for t in ts))
        self.torch.cuda.synchronize(self.device)

    def set_state(self, U, V, W):
        ts = [self._dev(t) for t in (U, V, W)]
        self.torch.cuda.current_stream(self.device).synchronize()
        gg3_set_state(self.ctx, *(t.data_ptr() for t in ts))
        self.torch.cuda.synchronize(self.device)

    def set_option(self, option, value):
        gg3_set_option(self.ctx, option, value)

    def step(self, n, dt):
        gg3_step(self.ctx, n, dt)

    def get_state_numpy(self):
        out = [self.torch.empty(self.shape, dtype=self.tdtype, device=self.device) for _ in range(3)]
        gg3_get_state(self.ctx, *(t.data_ptr() for t in out))
        self.torch.cuda.synchronize(self.device)
        return tuple(t.cpu().numpy() for t in out)

    @property
    def kernel(self) -> str:
        return KERNEL_NAMES[gg3_kernel_used(self.ctx)]

    @property
    def launches(self) -> int:
        return gg3_launches(self.ctx)

    @property
    def graph_captures(self) -> int:
        return gg3_graph_captures(self.ctx)

    def last_step_ms(self) -> float:
        return gg3_last_step_ms(self.ctx)

    def close(self):
        if self.ctx is not None:
            gg3_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def from_workload(wl, dtype="f64", device="cuda:0") -> Simulation3:
    """A Simulation3 holding a workloads.Workload3's tensor and initial state."""
    sim = Simulation3(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, wl.r, wl.d, wl.alpha, wl.c_r, dtype=dtype, device=device)
    sim.set_tensor(wl.tensor)
    sim.set_state(wl.U, wl.V, wl.W)
    return sim
