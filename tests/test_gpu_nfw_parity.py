"""GPU-vs-oracle parity of the pseudo-elliptical NFW body through the C ABI.  Same metric and
tolerances as the other lens models: fp64 1e-12, fp32 1e-5 of max|alpha| per component; mixed: rule kernels bit-exact
against the oracle's rule on an oracle-made fp32 map, end-to-end mask equal away from the thresholds, flagged pixels =
fp64 kernel's bits."""
import numpy as np
import pytest

from paper_1902_03252_b200 import workloads
import mixed_helpers as mh

pytestmark = pytest.mark.gpu

TOL_F64 = 1e-12
TOL_F32 = 1e-5


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_1902_03252_b200 import lt
    from oracle import lt_oracle_nfw as N
    from oracle import lt_oracle as O
    lt.lib()
    return torch, lt, N, O


def _gpu(torch, lt, W, mode, mixed=None, ws_out=None):
    L = torch.from_numpy(W.lenses).cuda()
    ws = lt.alloc_workspace(L.shape[0], W.nx, W.ny, mode)
    out = lt.lt_gradient_grid_nfw(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, mixed=mixed, workspace=ws)
    torch.cuda.synchronize()
    rc, bad = lt.lt_last_status(ws)
    assert rc == 0, (rc, bad)
    if ws_out is not None:
        ws_out.append(ws)
    return out.cpu().numpy()


def _err(a, ref):
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    return (np.abs(a.astype(np.float64) - ref).reshape(-1, 2).max(axis=0) / s).max()


@pytest.mark.parametrize("n", [96, 301, 512])
def test_cluster_full_grid(env, n):
    """2 cluster-scale + 62 galaxy-scale NFW halos; grids spanning several tiles with ragged tails"""
    torch, lt, N, O = env
    W = workloads.make_nfw(n_override=n)
    W = W._replace(ny=n - 7)
    ref = N.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    e64, e32 = _err(_gpu(torch, lt, W, lt.LT_FP64), ref), _err(_gpu(torch, lt, W, lt.LT_FP32), ref)
    print("nfw n", n, "fp64", e64, "fp32", e32)
    assert e64 < TOL_F64 and e32 < TOL_F32


def test_all_radial_regimes_against_the_quad_oracle(env):
    """Single lenses, points from R/rs = 1e-6 to 1e3 (the three branches of the kernel's w(u) and the neighbourhood of
    R = rs) against the __float128 instantiation; lt_gradient_points_nfw bit-equal to the grid kernel"""
    torch, lt, N, O = env
    rng = np.random.default_rng(21)
    for k in range(4):
        L = np.array([[rng.uniform(-10, 10), rng.uniform(-10, 10), rng.uniform(0, 0.3) if k else 0.0, rng.uniform(0, np.pi),
                       rng.uniform(0.05, 0.3), rng.uniform(1, 80)]])
        x = np.exp(rng.uniform(np.log(1e-6), np.log(1e3), 20000))
        x[:200] = 1.0 + rng.uniform(-1e-6, 1e-6, 200)
        x[200:400] = 0.5 + rng.uniform(-1e-6, 1e-6, 200)
        a = rng.uniform(0, 2 * np.pi, x.size)
        px, py = L[0, 0] + L[0, 5] * x * np.cos(a), L[0, 1] + L[0, 5] * x * np.sin(a)
        ref = N.gradient_points(L, px, py, N.QUAD)
        g = lt.lt_gradient_points_nfw(torch.from_numpy(L).cuda(), torch.from_numpy(np.stack([px, py], 1)).cuda()).cpu().numpy()
        assert np.isfinite(g).all()
        assert np.abs(g - ref).max() / np.abs(ref).max() < TOL_F64
    W = workloads.make_nfw(n_override=200)
    g64 = _gpu(torch, lt, W, lt.LT_FP64)
    i, j = rng.integers(0, W.nx, 20000), rng.integers(0, W.ny, 20000)      # > 4096: the thread-per-point kernel
    pts = torch.from_numpy(np.stack([W.x_min + i * W.dx, W.y_min + j * W.dx], axis=1)).cuda()
    gp = lt.lt_gradient_points_nfw(torch.from_numpy(W.lenses).cuda(), pts).cpu().numpy()
    assert np.array_equal(gp, g64[j, i])


def test_mixed_mode_and_edge_cases(env):
    torch, lt, N, O = env
    W = workloads.make_nfw(n_override=400)
    ws = []
    m = _gpu(torch, lt, W, lt.LT_MIXED, ws_out=ws)
    g64 = _gpu(torch, lt, W, lt.LT_FP64)
    g32 = _gpu(torch, lt, W, lt.LT_FP32)
    flags = lt.lt_mixed_last_flags(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy()
    ref = N.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    cat = N.as_rule_catalogue(W.lenses)
    mh.rule_parity(torch, lt, O, ref, cat, W, O.DEFAULT_MIXED)
    print("near-threshold fraction", mh.mask_agrees_away_from_thresholds(O, flags, ref, cat, W, O.DEFAULT_MIXED))
    f = flags != 0
    assert np.array_equal(m[f], g64[f]) and np.array_equal(m[~f], g32[~f].astype(np.float64))
    print("nfw mixed: flagged fraction", f.mean())
    # empty catalogue; pixel on a centre; domain error (rs <= 0)
    Z = W._replace(lenses=np.zeros((0, 6)), nx=40, ny=30)
    for mode in (lt.LT_FP64, lt.LT_FP32, lt.LT_MIXED):
        assert np.all(_gpu(torch, lt, Z, mode) == 0)
    one = workloads.Workload("centre", np.array([[0.0, 0.0, 0.1, 0.3, 0.2, 20.0]]), 0.0, 0.0, 0.5, 1, 1, 0)
    assert np.all(_gpu(torch, lt, one, lt.LT_FP64) == 0)
    bad = W.lenses.copy()
    bad[5, 5] = 0.0
    wsb = lt.alloc_workspace(len(bad), 8, 8, lt.LT_FP64)
    out = lt.lt_gradient_grid_nfw(torch.from_numpy(bad).cuda(), 0.0, 0.0, 1.0, 8, 8, workspace=wsb)
    rc, k = lt.lt_last_status(wsb)
    assert rc == lt.LT_ERR_BAD_LENS_PARAMS and k == 5 and torch.isnan(out).all()
    # host-buffer entry point
    hL = torch.from_numpy(W.lenses).pin_memory()
    hout = torch.empty((W.ny, W.nx, 2), dtype=torch.float64).pin_memory()
    wsh = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, lt.LT_FP64, host=True)
    lt.lt_gradient_grid_nfw_host(hL, W.x_min, W.y_min, W.dx, W.nx, W.ny, lt.LT_FP64, hout, wsh)
    torch.cuda.synchronize()
    assert np.array_equal(hout.numpy(), g64)
