"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol
include/wri.h declares, and validates arguments before touching CUDA."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2410_18429_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "wri.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(wri_[a-z_A-Z0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert {"wri_create", "wri_apply_M", "wri_apply_MH", "wri_lsqr_batch", "wri_lsqr_batch_host",
            "wri_destroy", "wri_strerror", "wri_workspace_bytes", "wri_set_workspace",
            "wri_lsqr_begin", "wri_lsqr_iterate", "wri_lsqr_end", "wri_lsqr_peek",
            "wri_set_model", "wri_launch_count", "wri_apply_S", "wri_apply_SH", "wri_lsqr_sf_batch",
            "wri_lsqr_sf_begin", "wri_lsqr_sf_batch_host", "wri_objective_gradient", "wri_lsqr_set_opts",
            "wri_misfit_sf", "wri_awri_step", "wri_set_receiver_mask",
            "wri_host_pipeline_bytes", "wri_set_host_pipeline", "wri_lsqr_batch_host_async",
            "wri_lsqr_sf_batch_host_async", "wri_host_wait", "wri_set_stencil",
            "wri_set_debug_opts", "wri_plan_info", "wri_objective_gradient_static"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_receiver_validation_precedes_cuda(lib):
    from paper_2410_18429_b200.binding import (wri_grid, wri_sponge, WRI_ERR_ARG,
                                               WRI_ERR_RECEIVER_DUP, WRI_ERR_RECEIVER_RANGE)
    om = np.array([31.4], dtype=np.float64)
    fake_m = C.c_void_p(256)     # never dereferenced on the host

    def create(rec, grid=(8, 8, 8), nb_max=4):
        rec = np.ascontiguousarray(rec, dtype=np.int32)
        h = C.c_void_p()
        rc = lib.wri_create(C.byref(h), wri_grid(*grid), 10.0, 1, om.ctypes.data_as(C.c_void_p), fake_m,
                            wri_sponge(2, 1.0, 2, 0x3F), len(rec), rec.ctypes.data_as(C.c_void_p), nb_max, None)
        assert not h.value or rc == 0
        if rc == 0:
            lib.wri_destroy(h)
        return rc

    assert create([[0, 0, 8]]) == WRI_ERR_RECEIVER_RANGE
    assert create([[-1, 0, 0]]) == WRI_ERR_RECEIVER_RANGE
    assert create([[1, 2, 3], [4, 4, 4], [1, 2, 3]]) == WRI_ERR_RECEIVER_DUP
    assert create([[1, 2, 3]], grid=(0, 8, 8)) == WRI_ERR_ARG
    assert create([[1, 2, 3]], nb_max=0) == WRI_ERR_ARG
    assert b"duplicate" in lib.wri_strerror(WRI_ERR_RECEIVER_DUP)
    assert lib.wri_workspace_bytes(None, 4, 0) == 0
    assert lib.wri_lsqr_iterate(None, 1) == WRI_ERR_ARG


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU a valid wri_create must fail with WRI_ERR_CUDA (never compute)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2410_18429_b200.binding import wri_grid, wri_sponge, WRI_ERR_CUDA
    om = np.array([31.4], dtype=np.float64)
    rec = np.array([[1, 2, 3]], dtype=np.int32)
    h = C.c_void_p()
    rc = lib.wri_create(C.byref(h), wri_grid(8, 8, 8), 10.0, 1, om.ctypes.data_as(C.c_void_p), C.c_void_p(256),
                        wri_sponge(2, 1.0, 2, 0x3F), 1, rec.ctypes.data_as(C.c_void_p), 4, None)
    assert rc == WRI_ERR_CUDA and not h.value
    assert b"CUDA" in lib.wri_strerror(rc)
