"""GPU-vs-oracle parity of the SIE body (the paper's Algorithm 1) through the C ABI.
Same metric and tolerances as tests/test_gpu_parity.py: fp64 1e-12, fp32 1e-5 of max|alpha| per component; mixed:
rule kernels bit-exact against the oracle's rule on an oracle-made fp32 map, end-to-end mask equal away from the
thresholds, flagged pixels = fp64 kernel's bits."""
import numpy as np
import pytest

from paper_1902_03252_b200 import workloads
import mixed_helpers as mh

pytestmark = pytest.mark.gpu

TOL_F64 = 1e-12
TOL_F32 = 1e-5
# the paper's own rule at its own pixel size; cluster-scale = b0 >= 1" (its two cluster halos have 28.8" and 14.1")
SIE_MIXED = (3.26, 0.0104 / 0.03, 6.0, 0.3, 1.0)


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_1902_03252_b200 import lt
    from oracle import lt_oracle_sie as S
    from oracle import lt_oracle as O
    lt.lib()
    return torch, lt, S, O


def _gpu(torch, lt, W, mode, mixed=None, ws_out=None):
    L = torch.from_numpy(W.lenses).cuda()
    ws = lt.alloc_workspace(L.shape[0], W.nx, W.ny, mode)
    out = lt.lt_gradient_grid_sie(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, mixed=mixed, workspace=ws)
    torch.cuda.synchronize()
    rc, bad = lt.lt_last_status(ws)
    assert rc == 0, (rc, bad)
    if ws_out is not None:
        ws_out.append(ws)
    return out.cpu().numpy()


def _err(a, ref, keep=None):
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    d = np.abs(a.astype(np.float64) - ref)
    if keep is not None:
        d = d[keep]
    return (d.reshape(-1, 2).max(axis=0) / s).max()


def _outside_patches(O, S, W):
    """Pixels outside the rule's DP centre patches: the set on which single precision is gated (R10;
    inside the patches the SIS direction theta/R amplifies the fp32 rounding of the coordinate, (A.65) P:876-880)."""
    z = np.zeros((W.ny, W.nx, 2), dtype=np.float32)
    return (O.mixed_flags(z, S.as_rule_catalogue(W.lenses), W.x_min, W.y_min, W.dx, mixed=SIE_MIXED) & 1) == 0


@pytest.mark.parametrize("n", [96, 203, 517])
def test_small_catalogue_full_grid(env, n):
    """2 + 30 halos on grids spanning several tiles with ragged tails in x and y."""
    torch, lt, S, O = env
    W = workloads.make_sie("small", n_override=n)
    W = W._replace(ny=n - 5)
    ref = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    g32 = _gpu(torch, lt, W, lt.LT_FP32)
    e64, e32 = _err(_gpu(torch, lt, W, lt.LT_FP64), ref), _err(g32, ref, _outside_patches(O, S, W))
    print("sie n", n, "fp64", e64, "fp32 outside patches", e32, "fp32 everywhere", _err(g32, ref))
    assert e64 < TOL_F64 and e32 < TOL_F32


def test_paper_benchmark_full_size_sampled(env):
    """The paper-like benchmark (6730^2, 702 halos) in the launch configuration bench.py times: sampled pixels (random,
    the pixels nearest every centre and their neighbours, the corners) against the oracle; lt_gradient_points_sie
    bit-equal to the grid kernel; the whole fp32 map against the oracle-checked fp64 map."""
    torch, lt, S, O = env
    W = workloads.make_sie("paper")
    g64 = _gpu(torch, lt, W, lt.LT_FP64)
    g32 = _gpu(torch, lt, W, lt.LT_FP32)
    rng = np.random.default_rng(3)
    i, j = rng.integers(0, W.nx, 20000), rng.integers(0, W.ny, 20000)
    ic = np.clip(np.round((W.lenses[:, 0] - W.x_min) / W.dx), 0, W.nx - 1).astype(np.int64)
    jc = np.clip(np.round((W.lenses[:, 1] - W.y_min) / W.dx), 0, W.ny - 1).astype(np.int64)
    i = np.concatenate([i, ic, np.clip(ic + 1, 0, W.nx - 1), ic, [0, W.nx - 1]])
    j = np.concatenate([j, jc, jc, np.clip(jc - 1, 0, W.ny - 1), [0, W.ny - 1]])
    px, py = W.x_min + i * W.dx, W.y_min + j * W.dx
    ref = S.gradient_points(W.lenses, px, py)
    s = np.abs(ref).max(axis=0)
    assert (np.abs(g64[j, i] - ref).max(axis=0) / s).max() < TOL_F64
    keep = _outside_patches(O, S, W)
    k = keep[j, i]
    assert (np.abs(g32[j, i].astype(np.float64) - ref)[k].max(axis=0) / s).max() < TOL_F32
    print("sie paper: fp32 sampled error inside patches (reported, not gated)",
          (np.abs(g32[j, i].astype(np.float64) - ref)[~k].max(axis=0) / s).max())
    pts = torch.from_numpy(np.stack([px, py], axis=1)).cuda()
    gp = lt.lt_gradient_points_sie(torch.from_numpy(W.lenses).cuda(), pts).cpu().numpy()
    assert np.array_equal(gp, g64[j, i])
    e = np.abs(g32.astype(np.float64) - g64)[keep].max(axis=0) / np.abs(g64).reshape(-1, 2).max(axis=0)
    print("sie paper: fp32 vs fp64 map outside patches", e, "patch fraction", 1 - keep.mean())
    assert e.max() < TOL_F32


def test_mixed_mode_follows_the_papers_rule(env):
    """The paper's mixed algorithm with its own constants at its own pixel size, on a window of the benchmark
    grid around the first cluster halo: rule kernels = oracle's rule on an oracle-made fp32 map (bit-exact), flagged pixels carry
    the fp64 kernel's bits, the others the fp32 value; the centre patch is inside the mask (Fig. 6); the error
    of every pixel meets the paper's criterion dx/(4 * 3.26)."""
    torch, lt, S, O = env
    W = workloads.make_sie("paper")
    i0 = int(round((W.lenses[0, 0] - W.x_min) / W.dx)) - 400
    j0 = int(round((W.lenses[0, 1] - W.y_min) / W.dx)) - 300
    W = W._replace(x_min=W.x_min + i0 * W.dx, y_min=W.y_min + j0 * W.dx, nx=900, ny=700)
    ws = []
    m = _gpu(torch, lt, W, lt.LT_MIXED, mixed=SIE_MIXED, ws_out=ws)
    g64 = _gpu(torch, lt, W, lt.LT_FP64)
    g32 = _gpu(torch, lt, W, lt.LT_FP32)
    flags = lt.lt_mixed_last_flags(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy()
    ref = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    cat = S.as_rule_catalogue(W.lenses)
    mh.rule_parity(torch, lt, O, ref, cat, W, SIE_MIXED)                      # the rule kernels on an oracle-made map
    print("near-threshold fraction", mh.mask_agrees_away_from_thresholds(O, flags, ref, cat, W, SIE_MIXED))
    f = flags != 0
    assert np.array_equal(m[f], g64[f]) and np.array_equal(m[~f], g32[~f].astype(np.float64))
    assert (flags[300 - 200:300 + 201, 400 - 200:400 + 201] & 1).all()       # 400 x 400 px DP patch
    assert np.abs(m - ref).max() <= W.dx / 4 / 3.26
    assert np.abs(m[f] - ref[f]).max() / np.abs(ref).max() < TOL_F64
    st = lt.lt_mixed_last_stats(ws[0])
    assert st["n_flagged"] == int(f.sum())
    print("sie mixed window: flagged fraction", f.mean(), st)


def test_edge_cases(env):
    torch, lt, S, O = env
    W = workloads.make_sie("small")
    Z = W._replace(lenses=np.zeros((0, 5)))
    for mode in (lt.LT_FP64, lt.LT_FP32, lt.LT_MIXED):
        assert np.all(_gpu(torch, lt, Z, mode) == 0)
    # pixel exactly on a lens centre: that lens contributes nothing (reading R5); eps = 0 lens; 1 x n and n x 1 grids
    L = W.lenses.copy()
    L[0, 0], L[0, 1] = 0.0, 0.0
    L[1, 2] = 0.0
    W2 = workloads.Workload("edge", L, -8.0, -8.0, 0.5, 40, 36, 0)          # pixel (16, 16) = (0, 0)
    ref = S.gradient_grid(W2.lenses, W2.x_min, W2.y_min, W2.dx, W2.nx, W2.ny)
    for mode, tol in ((lt.LT_FP64, TOL_F64), (lt.LT_FP32, TOL_F32)):
        a = _gpu(torch, lt, W2, mode)
        assert np.isfinite(a).all() and _err(a, ref, None if mode == lt.LT_FP64 else _outside_patches(O, S, W2)) < tol
    one = workloads.Workload("centre", L[0:1], 0.0, 0.0, 0.5, 1, 1, 0)
    assert np.all(_gpu(torch, lt, one, lt.LT_FP64) == 0) and np.all(_gpu(torch, lt, one, lt.LT_MIXED, mixed=SIE_MIXED) == 0)
    # fp32 cannot see "exactly on the centre" (its coordinates are tile-centre + offset): the SIS direction theta/R of a
    # rounding-level offset is arbitrary, the modulus stays <= b0 (1 + eps) and finite; the DP centre patch of the mixed
    # mode (above) is what the paper prescribes for these pixels ((A.65) P:876-880)
    a32 = _gpu(torch, lt, one, lt.LT_FP32)
    assert np.isfinite(a32).all() and np.hypot(*a32[0, 0]) <= L[0, 4] * (1 + L[0, 2]) * 1.001
    for nx, ny in ((1, 50), (70, 1)):
        W3 = W._replace(nx=nx, ny=ny)
        ref = S.gradient_grid(W3.lenses, W3.x_min, W3.y_min, W3.dx, nx, ny)
        assert _err(_gpu(torch, lt, W3, lt.LT_FP64), ref) < TOL_F64
        assert np.abs(_gpu(torch, lt, W3, lt.LT_MIXED) - ref).max() / np.abs(ref).max() < TOL_F32
    # domain error: |eps| >= 1
    bad = W.lenses.copy()
    bad[2, 2] = 1.5
    Lb = torch.from_numpy(bad).cuda()
    ws = lt.alloc_workspace(len(bad), 8, 8, lt.LT_FP64)
    out = lt.lt_gradient_grid_sie(Lb, 0.0, 0.0, 1.0, 8, 8, workspace=ws)
    rc, k = lt.lt_last_status(ws)
    assert rc == lt.LT_ERR_BAD_LENS_PARAMS and k == 2 and torch.isnan(out).all()


def test_host_buffer_entry_point(env):
    torch, lt, S, O = env
    W = workloads.make_sie("small")
    hL = torch.from_numpy(W.lenses).pin_memory()
    for mode, dt in ((lt.LT_FP64, torch.float64), (lt.LT_FP32, torch.float32)):
        hout = torch.empty((W.ny, W.nx, 2), dtype=dt).pin_memory()
        ws = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, mode, host=True)
        lt.lt_gradient_grid_sie_host(hL, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, hout, ws)
        torch.cuda.synchronize()
        assert np.array_equal(hout.numpy(), _gpu(torch, lt, W, mode))


@pytest.mark.parametrize("n_lens,nx,ny", [(37, 1400, 650), (702, 1500, 700), (1300, 1111, 600)])
def test_sie_records_from_the_constant_bank_give_the_same_bits(env, n_lens, nx, ny):
    """The SIE fp64 kernels (grid and quad) read their 48-byte records from __constant__ memory into uniform registers,
    eight lenses per iteration plus a lens-by-lens rest (37 = 4 groups + 5; 1300 records = two slot-loads that continue each
    other's sums); lt_set_tuning bit 5 keeps them in shared memory.  Same operations in the same order: fp64 and mixed maps
    bit-equal, through the host entry point too."""
    torch, lt, S, O = env
    rng = np.random.default_rng(500 + n_lens)
    L = np.stack([rng.uniform(-60, 60, n_lens), rng.uniform(-25, 25, n_lens), rng.uniform(0.0, 0.15, n_lens),
                  rng.uniform(0.0, np.pi, n_lens), rng.uniform(0.05, 0.3, n_lens)], axis=1)
    L[0, 4], L[1, 4] = 28.8, 14.1
    W = workloads.Workload("sie_const", L, -60.0, -25.0, 0.085, nx, ny, 0)
    res = {}
    for bit in (0, 32):
        try:
            lt.lt_set_tuning(single_launch=bit)
            res[bit] = (_gpu(torch, lt, W, lt.LT_FP64), _gpu(torch, lt, W, lt.LT_MIXED, mixed=SIE_MIXED))
        finally:
            lt.lt_set_tuning()
    assert np.array_equal(res[0][0], res[32][0]) and np.array_equal(res[0][1], res[32][1])
    assert np.isfinite(res[0][0]).all()
    hL = torch.from_numpy(L).pin_memory()
    hout = torch.full((ny, nx, 2), float("nan"), dtype=torch.float64).pin_memory()
    wsh = lt.alloc_workspace(n_lens, nx, ny, lt.LT_FP64, host=True)
    lt.lt_gradient_grid_sie_host(hL, W.x_min, W.y_min, W.dx, nx, ny, lt.LT_FP64, hout, wsh)
    torch.cuda.synchronize()
    assert np.array_equal(hout.numpy(), res[0][0])
