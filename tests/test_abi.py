"""Host-side checks of the C-ABI library (no GPU, no compute calls): it builds for sm_100a, loads, exports every
symbol include/lt_gradient.h declares, and its pure-host entry points behave as the header says."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1902_03252_b200.csrc import build
    build.build()
    from paper_1902_03252_b200 import lt
    return lt


def declared_functions():
    src = open(os.path.join(ROOT, "include", "lt_gradient.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lt_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported_and_bound(L):
    names = declared_functions()
    assert "lt_gradient_grid" in names and "lt_gradient_points" in names and len(names) >= 12
    lib = L.lib()
    for n in names:
        assert hasattr(lib, n), n
        assert n in L.SYMBOLS, n
    assert sorted(L.SYMBOLS) == names
    for n in names:
        if n not in ("lt_error_string", "lt_last_cuda_error"):
            assert hasattr(L, n), "python binding lacks " + n


def test_host_only_entry_points(L):
    assert L.lt_version() == 100
    p = L.lt_mixed_defaults()
    assert (p.m_max, p.patch_halfwidth_cluster, p.patch_halfwidth_galaxy, p.b0_cluster_threshold) == (3.26, 6.0, 0.3, 15.0)
    assert abs(p.c28 * 0.03 - 0.0104) < 1e-15                      # eq. 28 at the paper's 0.03"/px
    assert round(0.03 / p.m_max, 4) == 0.0092                      # eq. 25
    for code in range(-10, 1):
        assert L.lib().lt_error_string(code) not in (None, b"unknown error code")
    assert L.lib().lt_error_string(-99) == b"unknown error code"


def test_workspace_sizes(L):
    f = L.lt_workspace_bytes
    assert f(-1, 8, 8, 0) == 0 and f(8, 0, 8, 0) == 0 and f(8, 8, 8, 5) == 0 and f(70000, 8, 8, 0) == 0
    assert f(8, 65536, 32768, 0) == 0                              # nx*ny >= 2^31
    a, b, c = f(100, 1024, 1024, 0), f(100, 1024, 1024, 1), f(100, 1024, 1024, 2)
    assert a == b and a >= 256 + 100 * (128 + 64)
    assert c >= a + 1024 * 1024 * (1 + 8 + 4)                      # flag bytes + fp32 map + index list
    assert f(101, 1024, 1024, 2) >= c and f(100, 1025, 1024, 2) >= c
    assert f(0, 1, 1, 0) >= 256
    h = L.lt_host_workspace_bytes(100, 1024, 1024, 0)
    assert h >= a + 100 * 56 + 1024 * 1024 * 16
    assert L.lt_host_workspace_bytes(100, 1024, 1024, 1) >= b + 100 * 56 + 1024 * 1024 * 8


def test_argument_errors_need_no_gpu(L):
    """Argument validation happens before any CUDA call."""
    lib = L.lib()
    vp = ctypes.c_void_p
    assert lib.lt_gradient_grid(None, 4, 0.0, 0.0, 1.0, 8, 8, 0, None, vp(16), vp(16), 1 << 20, None) == -1
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 1.0, 0, 8, 0, None, vp(16), vp(16), 1 << 20, None) == -2
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 0.0, 8, 8, 0, None, vp(16), vp(16), 1 << 20, None) == -3
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, float("nan"), 1.0, 8, 8, 0, None, vp(16), vp(16), 1 << 20, None) == -3
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 3, None, vp(16), vp(16), 1 << 20, None) == -4
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 0, None, vp(16), vp(16), 100, None) == -5
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 0, None, vp(8), vp(16), 1 << 20, None) == -6
    bad = L.lt_mixed_params(-1.0, 0.3, 6.0, 0.3, 15.0)
    assert lib.lt_gradient_grid(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 2, ctypes.byref(bad), vp(16), vp(16), 1 << 20, None) == -7
    assert lib.lt_gradient_points(vp(16), 4, vp(16), -1, vp(16), vp(16), 1 << 20, None) == -2
    assert lib.lt_gradient_grid_noalloc(vp(16), 4097, 0.0, 0.0, 1.0, 8, 8, 0, vp(16), None) == -10   # LT_NOALLOC_MAX_LENSES
    assert lib.lt_gradient_grid_noalloc(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 2, vp(16), None) == -4
    assert lib.lt_set_tuning(-1, 0, 0, 0, 0, 0) == -2 and lib.lt_set_tuning(0, 0, 0, 0, 0, 0) == 0
    assert lib.lt_source_barycentres(vp(16), vp(16), vp(16), -1, 1.0, vp(16), None) == -2
    assert lib.lt_source_barycentres(vp(16), None, vp(16), 3, 1.0, vp(16), None) == -1
    assert lib.lt_source_barycentres(vp(16), vp(24), vp(16), 3, 1.0, vp(16), None) == -6
    assert lib.lt_source_barycentres(vp(16), vp(16), vp(16), 3, float("inf"), vp(16), None) == -3
    assert lib.lt_chi2(vp(16), vp(16), vp(16), 2, -1, vp(16), vp(16), 8, vp(16), vp(16), None) == -2
    assert lib.lt_chi2(vp(16), vp(16), vp(16), 0, 5, vp(16), vp(16), 8, vp(16), vp(16), None) == -2
    assert lib.lt_chi2(vp(16), vp(16), vp(16), 2, 5, vp(16), vp(16), 8, vp(16), None, None) == -1
    assert lib.lt_chi2(vp(8), vp(16), vp(16), 2, 5, vp(16), vp(16), 8, vp(16), vp(16), None) == -6


def test_binding_refuses_cpu_tensors(L):
    import torch
    with pytest.raises(TypeError):
        L.lt_gradient_grid(torch.zeros((2, 7), dtype=torch.float64), 0.0, 0.0, 1.0, 4, 4)


def test_product_does_not_import_oracle():
    """The product path may not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1902_03252_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "lt_oracle" not in src or fn == "workloads.py", fn
