"""lt_gradient_grid_noalloc (include/lt_gradient.h): the deflection map with the workspace in the library's built-in device
array, for callers that cannot allocate -- against the existing path, lt_gradient_grid with a caller-allocated workspace, on
calls in a row that share the array (different catalogues and grid sizes, so stale contents of the call before would
show).  Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the others.

Tolerances: those of tests/test_gpu_parity.py (fp64 1e-12, fp32 1e-5 of max|alpha| per component); the header also states
identical bits, which is checked too.
"""
import ctypes

import numpy as np
import pytest

from paper_1902_03252_b200 import workloads

pytestmark = pytest.mark.gpu

TOL_F64 = 1e-12
TOL_F32 = 1e-5


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_1902_03252_b200 import lt
    lt.lib()
    return torch, lt


def _err(a, ref):
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    return (np.abs(a.astype(np.float64) - ref.astype(np.float64)).reshape(-1, 2).max(axis=0) / s).max()


def _existing(torch, lt, W, nx, ny, mode):
    L = torch.from_numpy(W.lenses).cuda()
    ws = lt.alloc_workspace(L.shape[0], nx, ny, mode)
    out = lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, nx, ny, mode, workspace=ws)
    torch.cuda.synchronize()
    assert lt.lt_last_status(ws)[0] == 0
    return out.cpu().numpy()


def _noalloc(torch, lt, W, nx, ny, mode):
    L = torch.from_numpy(W.lenses).cuda()
    out = torch.full((ny, nx, 2), float("nan"), dtype=torch.float32 if mode == lt.LT_FP32 else torch.float64, device="cuda")
    torch.cuda.synchronize()
    lt.lt_gradient_grid_noalloc(L, W.x_min, W.y_min, W.dx, nx, ny, mode, out)
    torch.cuda.synchronize()
    assert lt.lt_noalloc_last_status() == (0, -1)
    return out.cpu().numpy()


def test_two_calls_in_a_row_match_the_existing_path(env):
    torch, lt = env
    # (config, nx, ny): 1000 lenses on a ragged grid of several tiles, then 100 lenses on another grid -- the second call
    # finds the first call's records, header and tables in the array; then the first again
    calls = [(3, 333, 201), (1, 200, 136), (3, 333, 201)]
    for mode, tol in ((lt.LT_FP64, TOL_F64), (lt.LT_FP32, TOL_F32)):
        for cfg, nx, ny in calls:
            W = workloads.make(cfg)
            ref = _existing(torch, lt, W, nx, ny, mode)
            got = _noalloc(torch, lt, W, nx, ny, mode)
            assert np.isfinite(got).all()
            assert _err(got, ref) < tol, (mode, cfg, _err(got, ref))
            assert np.array_equal(got, ref), (mode, cfg)          # the header's claim: identical bits


def test_against_the_oracle_on_config_0(env):
    torch, lt = env
    from oracle import lt_oracle as O
    W = workloads.make(0)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    assert _err(_noalloc(torch, lt, W, W.nx, W.ny, lt.LT_FP64), ref) < TOL_F64
    assert _err(_noalloc(torch, lt, W, W.nx, W.ny, lt.LT_FP32), ref) < TOL_F32


def test_limits_and_status(env):
    torch, lt = env
    lib = lt.lib()
    vp = ctypes.c_void_p
    # beyond the built-in scratch: a clear error before any CUDA call; mixed mode is refused
    assert lib.lt_gradient_grid_noalloc(vp(16), lt.LT_NOALLOC_MAX_LENSES + 1, 0.0, 0.0, 1.0, 8, 8, 0, vp(16), None) == -10
    assert b"LT_NOALLOC_MAX_LENSES" in lib.lt_error_string(-10)
    assert lib.lt_gradient_grid_noalloc(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 2, vp(16), None) == -4
    assert lib.lt_gradient_grid_noalloc(None, 4, 0.0, 0.0, 1.0, 8, 8, 0, vp(16), None) == -1
    assert lib.lt_gradient_grid_noalloc(vp(16), 4, 0.0, 0.0, 1.0, 8, 8, 0, vp(8), None) == -6
    # the maximum itself runs
    rng = np.random.default_rng(5)
    n = lt.LT_NOALLOC_MAX_LENSES
    lenses = np.stack([rng.uniform(-50, 50, n), rng.uniform(-50, 50, n), rng.uniform(0, 0.6, n), rng.uniform(0, np.pi, n),
                       rng.uniform(0.01, 1, n), rng.uniform(5, 50, n), rng.uniform(1, 10, n)], axis=1)
    L = torch.from_numpy(lenses).cuda()
    out = torch.empty((40, 70, 2), dtype=torch.float64, device="cuda")
    lt.lt_gradient_grid_noalloc(L, -50.0, -50.0, 1.0, 70, 40, lt.LT_FP64, out)
    ws = lt.alloc_workspace(n, 70, 40, lt.LT_FP64)
    ref = lt.lt_gradient_grid(L, -50.0, -50.0, 1.0, 70, 40, lt.LT_FP64, workspace=ws)
    torch.cuda.synchronize()
    assert lt.lt_noalloc_last_status() == (0, -1)
    assert torch.equal(out, ref)
    # the domain check of a call is its own: a bad lens is reported, the next good call is clean again
    bad = lenses[:300].copy()
    bad[257, 4] = -1.0                                            # rcore < 0
    lt.lt_gradient_grid_noalloc(torch.from_numpy(bad).cuda(), -50.0, -50.0, 1.0, 70, 40, lt.LT_FP64, out)
    assert lt.lt_noalloc_last_status() == (lt.LT_ERR_BAD_LENS_PARAMS, 257)
    lt.lt_gradient_grid_noalloc(L[:300].contiguous(), -50.0, -50.0, 1.0, 70, 40, lt.LT_FP64, out)
    assert lt.lt_noalloc_last_status() == (0, -1)
    assert torch.isfinite(out).all()
