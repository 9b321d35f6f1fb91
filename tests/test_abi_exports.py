"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol that
include/brmppi.h declares; host-only entry points behave as the header says.  No compute calls."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2508_05773_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "brmppi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(brmppi_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = declared_symbols()
    for required in ("brmppi_create", "brmppi_destroy", "brmppi_set_state", "brmppi_set_goal",
                     "brmppi_set_obstacles", "brmppi_solve", "brmppi_shift", "brmppi_step",
                     "brmppi_get_controls", "brmppi_workspace_bytes", "brmppi_strerror"):
        assert required in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = C.CDLL(lib_path)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/brmppi.h but not exported"


def test_python_binding_lists_the_same_names():
    from paper_2508_05773_b200 import brmppi
    assert sorted(brmppi.EXPORTS) == declared_symbols()


def test_host_only_calls(lib_path):
    import scenes
    from paper_2508_05773_b200 import brmppi
    lib = C.CDLL(lib_path)
    lib.brmppi_workspace_bytes.restype = C.c_size_t
    lib.brmppi_workspace_bytes.argtypes = [C.POINTER(brmppi.CParams)]
    lib.brmppi_strerror.restype = C.c_char_p
    p = scenes.default_params(K=16384, T=80)
    good = brmppi.make_cparams(p, 1, 8, 0)
    n = lib.brmppi_workspace_bytes(C.byref(good))
    assert 0 < n < (1 << 26)                       # a few hundred KB of partials, no per-sample data
    with_samples = brmppi.make_cparams(p, 1, 8, brmppi.FLAG_WRITE_SAMPLES)
    assert lib.brmppi_workspace_bytes(C.byref(with_samples)) >= n + 20 * p.K
    for bad_kw in (dict(K=0), dict(T=0), dict(T=100000), dict(dt=0.0), dict(lam=0.0), dict(L1=-1.0),
                   dict(sigma_v=-0.1), dict(v_min=1.0, v_max=-1.0), dict(delta_max=1.6)):
        bad = brmppi.make_cparams(p.with_(**bad_kw), 1, 8, 0)
        assert lib.brmppi_workspace_bytes(C.byref(bad)) == 0, bad_kw
    assert lib.brmppi_workspace_bytes(C.byref(brmppi.make_cparams(p, 1, 65, 0))) == 0
    assert lib.brmppi_workspace_bytes(C.byref(brmppi.make_cparams(p, 1, 8, 1 << 20))) == 0   # unknown flag
    assert lib.brmppi_workspace_bytes(None) == 0
    assert lib.brmppi_strerror(0) == b"ok"
    assert lib.brmppi_strerror(-4) == b"too many obstacles"
    assert lib.brmppi_strerror(-99) == b"unknown status"
    # NULL handling never dereferences
    assert lib.brmppi_destroy(None) == brmppi.ERR_NULL
    assert lib.brmppi_solve(None) == brmppi.ERR_NULL
    ctx = C.c_void_p()
    assert lib.brmppi_create(None, None, 0, None, C.byref(ctx)) == brmppi.ERR_NULL


def test_new_entry_points_validate_before_touching_cuda(lib_path):
    """brmppi_project / brmppi_hitch_filter: argument errors and the n = 0 no-op are decided on the host."""
    import numpy as np
    import scenes
    from paper_2508_05773_b200 import brmppi
    lib = C.CDLL(lib_path)
    fp = C.POINTER(C.c_float)
    lib.brmppi_project.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, fp, C.c_float,
                                   fp, fp, C.c_void_p, C.c_int]
    ones = (C.c_float * 10)(*([1.0] * 10))
    lo = (C.c_float * 10)(*([-1.0] * 10))
    assert lib.brmppi_project(None, 0, 8, None, None, None, ones, 0.1, lo, ones, None, 0) == brmppi.OK       # n = 0
    assert lib.brmppi_project(None, 0, 8, None, None, None, ones, 0.1, lo, ones, None, 1) == brmppi.OK
    assert lib.brmppi_project(None, 4, 9, None, None, None, ones, 0.1, lo, ones, None, 0) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_project(None, 4, 0, None, None, None, ones, 0.1, lo, ones, None, 0) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_project(None, -1, 8, None, None, None, ones, 0.1, lo, ones, None, 0) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_project(None, 4, 8, None, None, None, ones, -0.1, lo, ones, None, 0) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_project(None, 4, 8, None, None, None, ones, 0.1, lo, ones, None, 2) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_project(None, 4, 8, None, None, None, lo, 0.1, lo, ones, None, 0) == brmppi.ERR_INVALID_ARG   # w <= 0
    assert lib.brmppi_project(None, 4, 8, None, None, None, None, 0.1, lo, ones, None, 0) == brmppi.ERR_NULL
    assert lib.brmppi_project(None, 4, 8, None, None, None, ones, 0.1, lo, ones, None, 0) == brmppi.ERR_NULL        # A
    lib.brmppi_hitch_filter.argtypes = [C.c_void_p, C.POINTER(brmppi.CParams), C.c_int, fp, fp, fp, C.POINTER(C.c_int)]
    p = scenes.default_params()
    good = brmppi.make_cparams(p, 1, 0, 0)
    assert lib.brmppi_hitch_filter(None, C.byref(good), 0, None, None, None, None) == brmppi.OK                 # n = 0
    assert lib.brmppi_hitch_filter(None, None, 0, None, None, None, None) == brmppi.ERR_NULL
    assert lib.brmppi_hitch_filter(None, C.byref(good), -1, None, None, None, None) == brmppi.ERR_INVALID_ARG
    assert lib.brmppi_hitch_filter(None, C.byref(good), 3, None, None, None, None) == brmppi.ERR_NULL
    for kw in (dict(hitch_alpha=0.0), dict(hitch_alpha=1.1), dict(hitch_qv=0.0), dict(hitch_qdelta=-2.0), dict(dt=0.0)):
        bad = brmppi.make_cparams(p.with_(**kw), 1, 0, 0)
        assert lib.brmppi_hitch_filter(None, C.byref(bad), 0, None, None, None, None) == brmppi.ERR_INVALID_ARG, kw
    # the stabiliser's parameters are validated by brmppi_create only when it is switched on
    lib.brmppi_workspace_bytes.restype = C.c_size_t
    lib.brmppi_workspace_bytes.argtypes = [C.POINTER(brmppi.CParams)]
    assert lib.brmppi_workspace_bytes(C.byref(brmppi.make_cparams(p.with_(hitch_filter=0, hitch_alpha=0.0), 1, 8, 0))) > 0
    assert lib.brmppi_workspace_bytes(C.byref(brmppi.make_cparams(p.with_(hitch_filter=1, hitch_alpha=0.0), 1, 8, 0))) == 0
    assert lib.brmppi_workspace_bytes(C.byref(brmppi.make_cparams(p.with_(hitch_filter=2), 1, 8, 0))) == 0


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    import scenes
    from paper_2508_05773_b200 import brmppi
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        brmppi.Solver(scenes.default_params())


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2508_05773_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+[<\"].*oracle|liboracle", text, flags=re.M), \
                    f"{f} reaches into oracle/"
