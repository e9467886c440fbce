"""CPU-side checks of the boundary: libxy_b200.so builds, loads without a GPU, exports every
symbol include/xy.h declares, and validates its arguments.  No compute calls."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "xy.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(xy_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_mandated_calls():
    names = declared_functions()
    for f in ("xy_create", "xy_metropolis_sweep", "xy_overrelax_sweep", "xy_measure", "xy_pt_exchange"):
        assert f in names          # BASELINE.json north_star


def test_library_exports_every_declared_symbol(xy_mod):
    lib = xy_mod.load_library()
    names = declared_functions()
    assert len(names) >= 25
    for f in names:
        assert hasattr(lib, f), f"libxy_b200.so does not export {f}"
        assert f in xy_mod.SIGNATURES, f"binding.py has no prototype for {f}"
    assert sorted(xy_mod.SIGNATURES) == names


def test_create_validates_arguments(xy_mod):
    lib = xy_mod.load_library()
    b = np.linspace(0.44, 0.47, 8)
    pb = b.ctypes.data_as(C.POINTER(C.c_double))
    for L, R in ((7, 8), (12, 8), (0, 8), (-8, 8), (8, 0), (8, -1), (2048, 1)):
        assert not lib.xy_create(L, R, pb, 1), (L, R)
        assert lib.xy_last_error()
        assert lib.xy_state_bytes(L, R) == 0 and lib.xy_workspace_bytes(L, R) == 0
    assert not lib.xy_create(8, 8, None, 1)
    bad = b.copy(); bad[3] = np.nan
    assert not lib.xy_create(8, 8, bad.ctypes.data_as(C.POINTER(C.c_double)), 1)
    h = lib.xy_create(8, 8, pb, 1)
    assert h
    assert lib.xy_state_bytes(8, 8) == 8 * 512 * 4
    assert lib.xy_workspace_bytes(8, 8) >= 8 * 5 * 8
    # nothing is attached: every device call must refuse, not crash, and never compute on the CPU
    assert lib.xy_metropolis_sweep(h) == -3
    assert lib.xy_overrelax_sweep(h) == -3
    assert lib.xy_measure(h, None) == -3
    assert lib.xy_pt_exchange(h) == -3
    assert b"xy_attach" in lib.xy_last_error()
    n = (C.c_uint32 * 3)(5, 6, 7)
    assert lib.xy_set_counters(h, n) == 0
    m = (C.c_uint32 * 3)()
    assert lib.xy_get_counters(h, m) == 0 and list(m) == [5, 6, 7]
    v = C.c_int(0)
    assert lib.xy_get_option(h, 1, C.byref(v)) == 0 and 8 % v.value == 0
    assert lib.xy_set_option(h, 1, 3) == -1          # tile must divide L
    assert lib.xy_set_option(h, 99, 0) == -1
    lib.xy_destroy(h)
    lib.xy_destroy(None)


@pytest.mark.skipif(os.path.exists("/dev/nvidia0"), reason="a GPU is present")
def test_attach_without_gpu_fails_loudly(xy_mod):
    lib = xy_mod.load_library()
    b = np.linspace(0.44, 0.47, 8)
    h = lib.xy_create(8, 8, b.ctypes.data_as(C.POINTER(C.c_double)), 1)
    assert lib.xy_attach(h, None, None, None) == -4            # XY_ERR_NO_DEVICE
    assert b"no CPU fallback" in lib.xy_last_error()
    lib.xy_destroy(h)
    with pytest.raises(xy_mod.XYError):
        xy_mod.XY(8, 8, b, 1)


def test_input_recipe_matches_baseline_json():
    import json
    from paper_1211_0780_b200 import inputs
    cfgs = json.load(open(os.path.join(ROOT, "BASELINE.json")))["configs"]
    assert len(cfgs) == len(inputs.CONFIGS) == 5
    for text, c in zip(cfgs, inputs.CONFIGS):
        assert f"L={c.L}" in text and (f"R={c.R}" in text or f"{c.R} replicas" in text or f"{c.R}-replica" in text)
        assert str(c.mcs) + " MCS" in text
        b = inputs.betas_of(c)
        assert b.shape == (c.R,) and b[0] == c.beta_lo and abs(b[-1] - c.beta_hi) < 1e-15
        assert np.all(np.diff(b) > 0)
    assert inputs.HEADLINE.L == 160 and inputs.HEADLINE.R == 64


def test_create_accepts_every_documented_lattice_size(xy_mod):
    """include/xy.h: any L % 8 == 0 up to 1024.  Every such size must get a launchable tile (TY * L/8 within the
    kernel's launch bounds, shared memory within the opt-in limit): xy_create checks it and reports the tile."""
    lib = xy_mod.load_library()
    b = np.array([0.45])
    pb = b.ctypes.data_as(C.POINTER(C.c_double))
    for L in range(8, 1025, 8):
        h = lib.xy_create(L, 1, pb, 1)
        assert h, (L, lib.xy_last_error())
        ty, tz = C.c_int(0), C.c_int(0)
        assert lib.xy_get_option(h, 1, C.byref(ty)) == 0 and lib.xy_get_option(h, 2, C.byref(tz)) == 0
        assert ty.value >= 2 and L % ty.value == 0 and ty.value * (L // 8) <= 352, (L, ty.value)
        assert tz.value >= 2 and L % tz.value == 0
        lib.xy_destroy(h)


def test_build_is_stale_after_an_edit_to_any_kernel_header(tmp_path, monkeypatch):
    """The in-tree .so travels to the GPU box: the builder must never keep a library that was compiled from
    other sources.  Every file of csrc/ and include/ is a dependency (the colour-pass kernel xy_sweep.cuh was
    once missing from the list), and touching the CONTENT of any of them makes _stale() true."""
    import shutil
    from paper_1211_0780_b200 import build as B
    names = {os.path.basename(d) for d in B.dependencies()}
    for f in os.listdir(B.CSRC):
        if f.endswith((".cu", ".cuh")):
            assert f in names, f
    assert {"xy_sweep.cuh", "xy_api.cu", "xy_device.cuh", "xy_kernels.cuh", "xy.h"} <= names
    csrc, inc = tmp_path / "csrc", tmp_path / "include"
    shutil.copytree(B.CSRC, csrc)
    shutil.copytree(B.INCLUDE, inc)
    lib = tmp_path / "libxy_b200.so"
    monkeypatch.setattr(B, "CSRC", str(csrc))
    monkeypatch.setattr(B, "INCLUDE", str(inc))
    monkeypatch.setattr(B, "LIB_PATH", str(lib))
    monkeypatch.setattr(B, "HASH_PATH", str(lib) + ".hash")
    assert B._stale()                                    # no library yet
    lib.write_bytes(b"")
    (tmp_path / "libxy_b200.so.hash").write_text(B.source_hash() + "\n")
    assert not B._stale()
    for f in ("xy_sweep.cuh", "xy_kernels.cuh", "xy_device.cuh", "xy_api.cu"):
        with open(csrc / f, "a") as fh:
            fh.write("// edit\n")
        assert B._stale(), f
        (tmp_path / "libxy_b200.so.hash").write_text(B.source_hash() + "\n")
        assert not B._stale()
    with open(inc / "xy.h", "a") as fh:
        fh.write("/* edit */\n")
    assert B._stale()
    monkeypatch.setenv("XY_NVCC_EXTRA", "")
    (tmp_path / "libxy_b200.so.hash").write_text(B.source_hash() + "\n")
    monkeypatch.setenv("XY_NVCC_EXTRA", "-DXY_SWEEP_MIN_BLOCKS=3")
    assert B._stale(), "other compiler flags are another library"
