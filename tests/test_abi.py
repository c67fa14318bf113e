"""CPU-tier checks of the boundary: libgg.so builds, loads without a GPU, exports every symbol
include/gg.h declares, the binding covers the same set, and host-side argument validation works.
No compute call is made here (those need a device and live in test_gpu_parity.py)."""
import ctypes
import os
import re

import pytest

from paper_2006_01748_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header=os.path.join(ROOT, "include", "gg.h")):
    src = open(header).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gg_[a-z0-9_]+)\s*\(", src)))


TUNING_H = os.path.join(ROOT, "paper_2006_01748_b200", "csrc", "gg_tuning.h")


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for need in ("gg_create", "gg_set_tensor", "gg_set_state", "gg_step", "gg_get_state"):
        assert need in names
    # tuning knobs are not part of the installed interface
    text = open(os.path.join(ROOT, "include", "gg.h")).read()
    assert "_VARIANT" not in text and "gg_num_" not in text


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in declared_symbols() + declared_symbols(TUNING_H):
        assert hasattr(lib, name), f"libgg.so does not export {name}"


def test_binding_covers_exactly_the_header():
    assert sorted(binding.SIGNATURES) == declared_symbols()
    assert sorted(binding.TUNING_SIGNATURES) == declared_symbols(TUNING_H)
    for name in list(binding.SIGNATURES) + list(binding.TUNING_SIGNATURES):
        assert callable(getattr(binding, name)), f"binding lacks a function named {name}"


GG3_H = os.path.join(ROOT, "include", "gg3.h")


def declared_symbols3():
    src = re.sub(r"/\*.*?\*/", "", open(GG3_H).read(), flags=re.S)
    return sorted(set(re.findall(r"\b(gg3_[a-z0-9_]+)\s*\(", src)))


def test_3d_header_exports_and_binding_agree():
    from paper_2006_01748_b200 import binding3
    names = declared_symbols3()
    for need in ("gg3_create", "gg3_set_tensor", "gg3_set_state", "gg3_step", "gg3_get_state"):
        assert need in names
    lib = ctypes.CDLL(build.build())
    for name in names:
        assert hasattr(lib, name), f"libgg.so does not export {name}"
    assert sorted(binding3.SIGNATURES) == names
    for name in names:
        assert callable(getattr(binding3, name)), f"binding3 lacks a function named {name}"


def test_library_has_sm100a_code_and_tma():
    """The shipped cubin is for sm_100a and the stream kernel really uses TMA (UTMALDG in SASS)."""
    import subprocess
    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    out = subprocess.run([cuobjdump, "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run([cuobjdump, "-sass", "-fun",
                           "_ZN2gg14gg_step_streamIdLi2ELi4ELi8EEEvNS_10StreamArgsE", build.LIB],
                          capture_output=True, text=True).stdout
    assert "UTMALDG" in sass
    assert "DFMA" in sass


def test_create_validates_arguments():
    ok = binding.gg_create(8, 6, 0.5, 1.0, 10.0, 1e-3, 1.0)
    assert binding.gg_workspace_bytes(ok) >= 9 * 8 * 6 * 8
    binding.gg_destroy(ok)
    bad = [
        dict(nx=1, ny=8), dict(nx=8, ny=1), dict(h=0.0), dict(h=-1.0), dict(h=float("nan")),
        dict(dtype=7), dict(r=float("inf")),
    ]
    for kw in bad:
        args = dict(nx=8, ny=8, h=0.5, r=1.0, d=10.0, alpha=1e-3, c=1.0, dtype=binding.GG_F64)
        args.update(kw)
        with pytest.raises(binding.GGError) as e:
            binding.gg_create(**args)
        assert e.value.code in (binding.GG_ERR_ARG, binding.GG_ERR_UNSUPPORTED)
        assert str(e.value)


def test_create_xy_validates_mesh_sizes():
    ok = binding.gg_create_xy(2, 8, 6, 0.5, 0.25, 1.0, [2.0, 10.0], 1e-3, 1.0)
    assert binding.gg_workspace_bytes(ok) > 0
    binding.gg_destroy(ok)
    for dx, dy in ((0.0, 0.5), (0.5, -1.0), (float("nan"), 0.5), (0.5, float("inf"))):
        with pytest.raises(binding.GGError) as e:
            binding.gg_create_xy(1, 8, 6, dx, dy, 1.0, 10.0, 1e-3, 1.0)
        assert e.value.code == binding.GG_ERR_ARG


def test_calls_before_bind_are_state_errors():
    ctx = binding.gg_create(8, 8, 0.5, 1.0, 10.0, 1e-3, 1.0)
    try:
        with pytest.raises(binding.GGError) as e:
            binding.gg_step(ctx, 1, 1e-3)
        assert e.value.code == binding.GG_ERR_STATE
        with pytest.raises(binding.GGError) as e:
            binding.gg_set_state(ctx, 1, 1, 1)
        assert e.value.code == binding.GG_ERR_STATE
        with pytest.raises(binding.GGError) as e:
            binding.gg_bind(ctx, 0, 1 << 20, 0)
        assert e.value.code == binding.GG_ERR_ARG
        assert binding.gg_last_step_ms(ctx) < 0
        assert binding.gg_launches(ctx) == 0
    finally:
        binding.gg_destroy(ctx)


def test_options_validate():
    ctx = binding.gg_create(10, 8, 0.5, 1.0, 10.0, 1e-3, 1.0, binding.GG_F32)  # 40-byte rows
    try:
        assert binding.gg_kernel_used(ctx) == binding.GG_KERNEL_GENERIC  # AUTO: TMA needs 16 B rows
        with pytest.raises(binding.GGError) as e:
            binding.gg_set_option(ctx, binding.GG_OPT_KERNEL, binding.GG_KERNEL_STREAM)
        assert e.value.code == binding.GG_ERR_UNSUPPORTED
        with pytest.raises(binding.GGError):
            binding.gg_set_option(ctx, 99, 0)
        with pytest.raises(binding.GGError):
            binding.gg_set_option(ctx, binding.GG_OPT_STREAM_VARIANT, binding.gg_num_stream_variants())
        binding.gg_set_option(ctx, binding.GG_OPT_GRAPH, 0)
    finally:
        binding.gg_destroy(ctx)
    ctx = binding.gg_create(12, 8, 0.5, 1.0, 10.0, 1e-3, 1.0, binding.GG_F32)
    try:
        assert binding.gg_kernel_used(ctx) == binding.GG_KERNEL_RESIDENT  # AUTO: tiny grids stay on chip
    finally:
        binding.gg_destroy(ctx)


def test_noalloc_entry_point_validates_before_touching_the_device():
    """gg_diagnostics_noalloc checks its arguments before any CUDA call, so the refusals can be
    seen without a GPU: a batch beyond the built-in scratch, NULL arrays, bad sizes."""
    nb = binding.GG_NOALLOC_MAX_BATCH
    fake = 4096                                         # never dereferenced: validation fails first
    with pytest.raises(binding.GGError) as e:
        binding.gg_diagnostics_noalloc(fake, fake, fake, nb + 1, 8, 8, binding.GG_F64, 0.1, fake, 0)
    assert e.value.code == binding.GG_ERR_ARG and "GG_NOALLOC_MAX_BATCH" in str(e.value)
    for args in ((0, fake, fake, 1, 8, 8, binding.GG_F64, 0.1, fake), (fake, fake, fake, 1, 8, 8, binding.GG_F64, 0.1, 0),
                 (fake, fake, fake, 0, 8, 8, binding.GG_F64, 0.1, fake), (fake, fake, fake, 1, 8, 0, binding.GG_F64, 0.1, fake),
                 (fake, fake, fake, 1, 8, 8, binding.GG_F64, -1.0, fake), (fake + 4, fake, fake, 1, 8, 8, binding.GG_F64, 0.1, fake)):
        with pytest.raises(binding.GGError) as e:
            binding.gg_diagnostics_noalloc(*args, 0)
        assert e.value.code == binding.GG_ERR_ARG and binding.gg_noalloc_last_error()
    with pytest.raises(binding.GGError) as e:
        binding.gg_diagnostics_noalloc(fake, fake, fake, 1, 8, 8, 9, 0.1, fake, 0)
    assert e.value.code == binding.GG_ERR_UNSUPPORTED


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(RuntimeError):
        binding.Simulation(8, 8, 0.5, 1.0, 10.0, 1e-3, 1.0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2006_01748_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "gg_oracle" not in text, f
