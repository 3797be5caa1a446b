"""The C-ABI library loads without a GPU, exports every symbol include/vr.h declares, and rejects
bad arguments before touching the device (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1008_0135_b200 import build as vr_build
from paper_1008_0135_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def vr():
    vr_build.build()
    from paper_1008_0135_b200 import vr as binding
    binding.lib()
    return binding


def declared_symbols(headers=("vr.h", "vr_measure.h")):
    names = set()
    for h in headers:
        text = open(os.path.join(ROOT, "include", h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(vr_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_exported(vr):
    names = declared_symbols()
    assert set(names) == set(vr.SYMBOLS), (names, vr.SYMBOLS)
    L = C.CDLL(vr.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} is declared in include/vr.h but not exported"


def test_experiment_builds_never_replace_the_product_library(monkeypatch):
    """A VR_DEFINES build goes to a file of its own, keyed by the defines; every csrc file is a dependency."""
    monkeypatch.delenv("VR_DEFINES", raising=False)
    product = vr_build.lib_path()
    assert product == vr_build.LIB and os.path.basename(product) == "libvr_b200.so"
    monkeypatch.setenv("VR_DEFINES", "-DVR_EXP_MORTON")
    a = vr_build.lib_path()
    monkeypatch.setenv("VR_DEFINES", "-DVR_CTA_H=4 -DVR_CAST_MINBLOCKS=14")
    b = vr_build.lib_path()
    assert len({product, a, b}) == 3 and all(p.endswith(".so") for p in (a, b))
    names = {os.path.basename(p) for p in vr_build.deps()}
    assert {"vr_api.cu", "kernels.cuh", "sampler.cuh", "slab.cuh", "plan.h", "vr.h"} <= names


def test_product_header_stays_small():
    """include/vr.h is the product boundary (SURVEY.md section 8(b) + the NEXT rows); measurement and test aids live in
    include/vr_measure.h."""
    product = declared_symbols(("vr.h",))
    aids = declared_symbols(("vr_measure.h",))
    assert len(product) <= 24, product
    assert set(aids) == {"vr_measure", "vr_measure_units", "vr_get_stage_ms", "vr_volume_info", "vr_export_linear"}
    assert not set(product) & set(aids)


def test_last_error_never_null(vr):
    assert isinstance(vr.vr_last_error(), str)


def test_null_and_range_checks_without_device(vr):
    L = vr.lib()
    out = C.c_void_p()
    dims = (C.c_int * 3)(8, 8, 8)
    assert L.vr_create_volume(None, None, C.byref(out)) == vr.VR_ERR_INVALID_ARG
    assert L.vr_create_volume(dims, None, C.byref(out)) == vr.VR_ERR_INVALID_ARG
    bad = (C.c_int * 3)(8, 0, 8)
    assert L.vr_create_volume(bad, C.c_void_p(16), C.byref(out)) == vr.VR_ERR_INVALID_ARG
    assert "dim" in vr.vr_last_error()
    assert L.vr_set_stream(None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_bricks(None, 1, 1, 1) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_subcube(None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_channel_mask(None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_transfer_function(None, None, 0.0, 1.0) == vr.VR_ERR_INVALID_ARG
    cam = vr.camera_from_spec(wl.orbit_camera((8, 8, 8), 30, 20, wl.PROJ_ORTHO))
    assert L.vr_render(None, C.byref(cam), 8, 8, 1.0, 0, 0.0, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_render_to_host(None, C.byref(cam), 8, 8, 1.0, 0, 0.0, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_render_to_host_async(None, C.byref(cam), 8, 8, 1.0, 0, 0.0, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_wait_frames(None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_measure(None, C.byref(cam), 8, 8, 1.0, 0, 0.0, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_measure_units(None, C.byref(cam), 8, 8, 1.0, 0, 0.0, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_empty_space_skipping(None, 1) == vr.VR_ERR_INVALID_ARG
    assert L.vr_get_skip_info(None, None, None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_set_slab_staging(None, 1) == vr.VR_ERR_INVALID_ARG
    assert L.vr_get_slab_info(None, None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_plan_slab(None, None, C.byref(cam), 8, 8, 1.0, None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_volume_info(None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_export_linear(None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_volume_range(None, None, None) == vr.VR_ERR_INVALID_ARG
    assert L.vr_volume_histogram(None, 16, 0.0, 1.0, None, None) == vr.VR_ERR_INVALID_ARG
    L.vr_destroy_volume(None)     # no-op


def test_plan_rejects_bad_cameras(vr):
    dims, bricks = (16, 16, 16), (2, 2, 2)
    good = wl.orbit_camera(dims, 30, 20, wl.PROJ_PERSP)
    vr.vr_plan_bricks(dims, bricks, vr.camera_from_spec(good), 32, 32)
    skew = np.array(good.view, dtype=np.float32).copy()
    skew[0, 0] += 0.01
    with pytest.raises(vr.VrError) as e:
        vr.vr_plan_bricks(dims, bricks, vr.make_camera(skew, wl.PROJ_PERSP, 45.0, 1.0), 32, 32)
    assert e.value.status == vr.VR_ERR_INVALID_ARG and "orthonormal" in str(e.value)
    for kw in (dict(projection=wl.PROJ_PERSP, fovy_deg=0.0), dict(projection=wl.PROJ_PERSP, fovy_deg=180.0),
               dict(projection=wl.PROJ_ORTHO, ortho_half_h=0.0), dict(projection=7)):
        with pytest.raises(vr.VrError):
            vr.vr_plan_bricks(dims, bricks, vr.make_camera(good.view, **kw), 32, 32)
    with pytest.raises(vr.VrError):
        vr.vr_plan_bricks(dims, (32, 1, 1), vr.camera_from_spec(good), 32, 32)   # b_a > n_a
    with pytest.raises(vr.VrError):
        vr.vr_plan_bricks(dims, (16, 16, 16), vr.camera_from_spec(good), 32, 32)  # > VR_MAX_BRICKS
    with pytest.raises(vr.VrError):
        vr.vr_plan_bricks(dims, bricks, vr.camera_from_spec(good), 0, 32)


def test_no_device_is_an_error_not_a_fallback(vr):
    """Without a CUDA device a compute call must fail with VR_ERR_CUDA / VR_ERR_OOM, never succeed."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = vr.lib()
    out = C.c_void_p()
    dims = (C.c_int * 3)(8, 8, 8)
    st = L.vr_create_volume(dims, C.c_void_p(256), C.byref(out))
    assert st in (vr.VR_ERR_CUDA, vr.VR_ERR_OOM)
    assert not out.value
    assert vr.vr_last_error()
