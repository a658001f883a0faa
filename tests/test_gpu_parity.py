"""GPU-vs-oracle parity through the C ABI (python binding = marshalling only).  Run on the B200 box: pytest -m gpu.

Metric (R9): per component, max over pixels of |GPU - oracle| / max over pixels of |alpha_oracle|.
Tolerances: fp64 1e-12 (north star); fp32 1e-5 (north star's example, = the SP accuracy the
paper deems sufficient away from the DP set); mixed: flagged pixels bit-equal to the fp64 mode and <= 1e-12 of the
oracle, unflagged pixels == fp32 mode widened.
"""
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
    from oracle import lt_oracle as O
    lt.lib()
    return torch, lt, O


def _gpu_map(torch, lt, W, mode, mixed=None, nx=None, ny=None, ws_out=None):
    nx = W.nx if nx is None else nx
    ny = W.ny if ny is None else ny
    L = torch.from_numpy(W.lenses).cuda()
    ws = lt.alloc_workspace(L.shape[0], nx, ny, mode)
    out = lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, nx, ny, mode, mixed=mixed, workspace=ws)
    torch.cuda.synchronize()
    rc, bad = lt.lt_last_status(ws)
    assert rc == 0, (rc, bad)
    if ws_out is not None:
        ws_out.append(ws)
    return out.cpu().numpy()


def _err(a, ref):
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    return (np.abs(a.astype(np.float64) - ref).reshape(-1, 2).max(axis=0) / s).max()


def test_cfg0_fp64_fp32_full_grid(env):
    torch, lt, O = env
    W = workloads.make(0)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    assert _err(_gpu_map(torch, lt, W, lt.LT_FP64), ref) < TOL_F64
    assert _err(_gpu_map(torch, lt, W, lt.LT_FP32), ref) < TOL_F32


@pytest.mark.parametrize("cfg,n", [(1, 200), (2, 136), (4, 2048)])
def test_reduced_grids_span_tiles_and_ragged_tail(env, cfg, n):
    """Catalogues of configs 1, 2 (coarser grid of the same extent: several tiles, ragged tails in x and y) and the
    stress config 4 on a window of its full-resolution grid around lens centres."""
    torch, lt, O = env
    W = workloads.make(cfg, n_override=n if cfg != 4 else None)
    if cfg == 4:
        # 300 x 77 window of the 2048^2 grid whose lower-left corner sits 20 px left/below lens 5's nearest pixel
        i0 = int(round((W.lenses[5, 0] - W.x_min) / W.dx)) - 20
        j0 = int(round((W.lenses[5, 1] - W.y_min) / W.dx)) - 20
        W = W._replace(x_min=W.x_min + i0 * W.dx, y_min=W.y_min + j0 * W.dx, nx=300, ny=77)
    else:
        W = W._replace(nx=n, ny=n - 3)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    e64 = _err(_gpu_map(torch, lt, W, lt.LT_FP64), ref)
    e32 = _err(_gpu_map(torch, lt, W, lt.LT_FP32), ref)
    print("cfg", cfg, "fp64 err", e64, "fp32 err", e32)
    assert e64 < TOL_F64
    assert e32 < TOL_F32


@pytest.mark.parametrize("ppt64,ppt32,chunk", [(1, 1, 0), (2, 2, 3), (4, 4, 64), (1, 4, 1)])
def test_launch_configurations_agree(env, ppt64, ppt32, chunk):
    """Every pixels-per-thread / lens-chunk variant gives the same fp64 bits and fp32 within tolerance."""
    torch, lt, O = env
    W = workloads.make(1, n_override=97)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    base = _gpu_map(torch, lt, W, lt.LT_FP64)
    try:
        lt.lt_set_tuning(ppt64, ppt32, chunk, chunk, 0)
        a = _gpu_map(torch, lt, W, lt.LT_FP64)
        b = _gpu_map(torch, lt, W, lt.LT_FP32)
    finally:
        lt.lt_set_tuning()
    assert np.array_equal(a, base)
    assert _err(a, ref) < TOL_F64 and _err(b, ref) < TOL_F32


@pytest.mark.parametrize("n_lens,nx,ny", [(100, 1500, 700), (449, 1300, 333), (1000, 1111, 600)])
def test_records_from_the_constant_bank_give_the_same_bits(env, n_lens, nx, ny):
    """The fp64 kernels read the lens records from __constant__ memory where the call allows it (one slot of 448 dPIE
    records: 449 and 1000 lenses take two and three launches that continue each other's sums); lt_set_tuning bit 5 keeps
    them in shared memory.  Same operations in the same order: fp64 and mixed maps bit-equal, on grids with whole waves
    and a ragged rest, also when two streams use the slot alternately."""
    torch, lt, O = env
    L = workloads.random_catalogue(31 + n_lens, n_lens, L=60.0)
    W = workloads.Workload("const", L, -60.0, -25.0, 0.085, nx, ny, 0)
    res = {}
    for bit in (0, 32):
        try:
            lt.lt_set_tuning(single_launch=bit)
            res[bit] = (_gpu_map(torch, lt, W, lt.LT_FP64), _gpu_map(torch, lt, W, lt.LT_MIXED))
        finally:
            lt.lt_set_tuning()
    assert np.array_equal(res[0][0], res[32][0]) and np.array_equal(res[0][1], res[32][1])
    assert lt.lt_last_launch_count() >= 1
    # two streams, two different catalogues, interleaved calls: each map equals its single-stream result
    L2 = workloads.random_catalogue(77, n_lens, L=60.0)
    d1, d2 = torch.from_numpy(L).cuda(), torch.from_numpy(L2).cuda()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    ref2 = lt.lt_gradient_grid(d2, W.x_min, W.y_min, W.dx, nx, ny, lt.LT_FP64).cpu().numpy()
    outs = []
    for rep in range(3):
        a = lt.lt_gradient_grid(d1, W.x_min, W.y_min, W.dx, nx, ny, lt.LT_FP64, stream=s1)
        b = lt.lt_gradient_grid(d2, W.x_min, W.y_min, W.dx, nx, ny, lt.LT_FP64, stream=s2)
        outs.append((a, b))
    torch.cuda.synchronize()
    for a, b in outs:
        assert np.array_equal(a.cpu().numpy(), res[0][0]) and np.array_equal(b.cpu().numpy(), ref2)
    # the host entry point: the map goes straight into pinned host memory; with several slot-loads the partial sums stay in
    # the call's device staging buffer and only the last launch writes across PCIe
    hL = torch.from_numpy(L).pin_memory()
    for mode, k in ((lt.LT_FP64, 0), (lt.LT_MIXED, 1)):
        hout = torch.full((ny, nx, 2), float("nan"), dtype=torch.float64).pin_memory()
        wsh = lt.alloc_workspace(n_lens, nx, ny, mode, host=True)
        lt.lt_gradient_grid_host(hL, W.x_min, W.y_min, W.dx, nx, ny, mode, hout, wsh)
        torch.cuda.synchronize()
        assert np.array_equal(hout.numpy(), res[0][k])


def test_oversized_chunk_request_is_clamped(env):
    """lt_set_tuning(chunk64 = chunk32 = 65536) with 4096 lenses: the wanted chunk exceeds what fits beside each kernel's
    own static shared memory (the range-reduction tables) under the opt-in limit; the library clamps it per kernel instead
    of failing the launch, and the map does not change (fp64 bit-equal, all three modes run)."""
    torch, lt, O = env
    L = workloads.random_catalogue(11, 4096, L=80.0)
    W = workloads.Workload("many", L, -80.0, -80.0, 2.5, 64, 40, 11)
    base = _gpu_map(torch, lt, W, lt.LT_FP64)
    try:
        lt.lt_set_tuning(0, 0, 65536, 65536, 0)
        a = _gpu_map(torch, lt, W, lt.LT_FP64)
        b = _gpu_map(torch, lt, W, lt.LT_FP32)
        m = _gpu_map(torch, lt, W, lt.LT_MIXED)
    finally:
        lt.lt_set_tuning()
    assert np.array_equal(a, base)
    s = np.abs(base).max()
    assert np.abs(b.astype(np.float64) - base).max() / s < TOL_F32 and np.abs(m - base).max() / s < TOL_F32


@pytest.mark.parametrize("nx,ny,ctas", [(1500, 1111, 0), (1027, 2049, 1), (4096, 300, 2), (129, 4100, 0)])
def test_wave_split_covers_every_pixel_once(env, nx, ny, ctas):
    """The launch plan (whole waves of the widest variant, ragged rest to the finer ones: lt_api.cu launch_waves)
    writes every pixel exactly as the single-launch plan does: fp64 bit-equal, fp32 within tolerance, no pixel left
    unwritten (the output is poisoned with NaN first)."""
    torch, lt, O = env
    W = workloads.make(0)
    L = torch.from_numpy(W.lenses[:3].copy()).cuda()
    x_min, y_min, dx = -40.0, -31.0, 0.05
    res = {}
    for single in (1, 0):
        for mode, dt in ((lt.LT_FP64, torch.float64), (lt.LT_FP32, torch.float32)):
            out = torch.full((ny, nx, 2), float("nan"), dtype=dt, device="cuda")
            try:
                lt.lt_set_tuning(0, 0, 0, 0, ctas, single)
                lt.lt_gradient_grid(L, x_min, y_min, dx, nx, ny, mode, out=out)
                n_launch = lt.lt_last_launch_count()
            finally:
                lt.lt_set_tuning()
            torch.cuda.synchronize()
            assert not torch.isnan(out).any()
            assert n_launch == 2 if single else n_launch >= 2
            res[(single, mode)] = out.cpu().numpy()
    assert np.array_equal(res[(0, lt.LT_FP64)], res[(1, lt.LT_FP64)])
    s = np.abs(res[(1, lt.LT_FP64)]).max()
    assert np.abs(res[(0, lt.LT_FP32)].astype(np.float64) - res[(1, lt.LT_FP64)]).max() / s < TOL_F32
    # a sample of pixels against the oracle (the rest is covered by the equality above)
    rng = np.random.default_rng(7)
    i, j = rng.integers(0, nx, 500), rng.integers(0, ny, 500)
    ref = O.gradient_points(W.lenses[:3], x_min + i * dx, y_min + j * dx)
    assert np.abs(res[(0, lt.LT_FP64)][j, i] - ref).max() / np.abs(ref).max() < TOL_F64


def test_full_size_cfg1_sampled_and_points(env):
    """BASELINE config 1 at full size, in the launch configuration bench.py times: sampled pixels (random + the pixels
    nearest every lens centre) against the oracle, and lt_gradient_points against the grid kernel (bit-equal)."""
    torch, lt, O = env
    W = workloads.make(1)
    g64 = _gpu_map(torch, lt, W, lt.LT_FP64)
    g32 = _gpu_map(torch, lt, W, lt.LT_FP32)
    rng = np.random.default_rng(42)
    i = rng.integers(0, W.nx, 20000)
    j = rng.integers(0, W.ny, 20000)
    ic = np.clip(np.round((W.lenses[:, 0] - W.x_min) / W.dx), 0, W.nx - 1).astype(np.int64)
    jc = np.clip(np.round((W.lenses[:, 1] - W.y_min) / W.dx), 0, W.ny - 1).astype(np.int64)
    i = np.concatenate([i, ic, np.clip(ic + 1, 0, W.nx - 1), [0, W.nx - 1]])
    j = np.concatenate([j, jc, jc, [0, W.ny - 1]])
    px, py = W.x_min + i * W.dx, W.y_min + j * W.dx
    ref = O.gradient_points(W.lenses, px, py)
    s = np.abs(ref).max(axis=0)
    assert (np.abs(g64[j, i] - ref).max(axis=0) / s).max() < TOL_F64
    assert (np.abs(g32[j, i].astype(np.float64) - ref).max(axis=0) / s).max() < TOL_F32
    pts = torch.from_numpy(np.stack([px, py], axis=1)).cuda()
    gp = lt.lt_gradient_points(torch.from_numpy(W.lenses).cuda(), pts).cpu().numpy()
    assert np.array_equal(gp, g64[j, i])
    # the whole fp32 map against the (now oracle-checked) fp64 map
    assert _err(g32, g64) < TOL_F32


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_size_configs_sampled(env, cfg):
    """BASELINE configs 2, 3 and 4 (the precision stress case) at full size: 20000 random pixels plus the pixels nearest
    every lens centre against the oracle in fp64 and fp32; the whole fp32 map against the oracle-checked fp64 map; the
    whole mixed map = fp64 bits on flagged pixels, fp32 value elsewhere."""
    torch, lt, O = env
    W = workloads.make(cfg)
    ws = []
    g64 = _gpu_map(torch, lt, W, lt.LT_FP64)
    g32 = _gpu_map(torch, lt, W, lt.LT_FP32)
    rng = np.random.default_rng(100 + cfg)
    i, j = rng.integers(0, W.nx, 20000), rng.integers(0, W.ny, 20000)
    ic = np.clip(np.round((W.lenses[:, 0] - W.x_min) / W.dx), 0, W.nx - 1).astype(np.int64)
    jc = np.clip(np.round((W.lenses[:, 1] - W.y_min) / W.dx), 0, W.ny - 1).astype(np.int64)
    i = np.concatenate([i, ic, np.clip(ic - 1, 0, W.nx - 1), [0, W.nx - 1]])
    j = np.concatenate([j, jc, np.clip(jc + 1, 0, W.ny - 1), [W.ny - 1, 0]])
    ref = O.gradient_points(W.lenses, W.x_min + i * W.dx, W.y_min + j * W.dx)
    s = np.abs(ref).max(axis=0)
    e64 = (np.abs(g64[j, i] - ref).max(axis=0) / s).max()
    e32 = (np.abs(g32[j, i].astype(np.float64) - ref).max(axis=0) / s).max()
    smax = np.abs(g64).reshape(-1, 2).max(axis=0)
    e32_map = (np.abs(g32.astype(np.float64) - g64).reshape(-1, 2).max(axis=0) / smax).max()
    print("cfg", cfg, "sampled fp64", e64, "fp32", e32, "fp32 map vs fp64 map", e32_map)
    assert e64 < TOL_F64 and e32 < TOL_F32 and e32_map < TOL_F32
    m = _gpu_map(torch, lt, W, lt.LT_MIXED, ws_out=ws)
    f = lt.lt_mixed_last_flags(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy() != 0
    st = lt.lt_mixed_last_stats(ws[0])
    assert st["n_flagged"] == int(f.sum())
    assert np.array_equal(m[f], g64[f]) and np.array_equal(m[~f], g32[~f].astype(np.float64))


def test_mixed_mode_follows_the_rule(env):
    """Mixed mode on config 0 and on the paper-regime variant of config 1 (reduced grid): the rule kernels equal the
    oracle's rule bit for bit on an oracle-made fp32 map; the end-to-end mask equals the oracle's mask away from the
    thresholds; flagged pixels carry the fp64 kernel's bits, unflagged pixels the fp32 kernel's value widened; the
    stats agree with the mask."""
    torch, lt, O = env
    for W in (workloads.make(0), workloads.make(1, paper_regime=True, n_override=333)):
        ws = []
        m = _gpu_map(torch, lt, W, lt.LT_MIXED, ws_out=ws)
        g64 = _gpu_map(torch, lt, W, lt.LT_FP64)
        g32 = _gpu_map(torch, lt, W, lt.LT_FP32)
        flags = lt.lt_mixed_last_flags(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy()
        ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
        mh.rule_parity(torch, lt, O, ref, W.lenses, W, O.DEFAULT_MIXED)          # the rule kernels on an oracle-made map
        # the end-to-end call ran the same kernels on its own fp32 map ...
        c3 = torch.from_numpy(np.ascontiguousarray(W.lenses[:, [0, 1, 6]])).cuda()
        again, _ = lt.lt_mixed_rule(torch.from_numpy(g32).cuda(), W.x_min, W.y_min, W.dx, c3)
        assert np.array_equal(flags, again.cpu().numpy())
        # ... and its mask is the oracle's wherever no criterion sits on a threshold (R18)
        print(W.name, "near-threshold fraction", mh.mask_agrees_away_from_thresholds(O, flags, ref, W.lenses, W, O.DEFAULT_MIXED))
        st = lt.lt_mixed_last_stats(ws[0])
        assert st["n_flagged"] == int((flags != 0).sum())
        assert st["n_patch"] == int((flags & 1).astype(bool).sum())
        assert st["n_eq25"] == int((flags & 2).astype(bool).sum())
        assert st["n_eq28"] == int((flags & 4).astype(bool).sum())
        f = flags != 0
        assert np.array_equal(m[f], g64[f])
        assert np.array_equal(m[~f], g32[~f].astype(np.float64))
        s = np.abs(ref).max()
        if f.any():
            assert np.abs(m[f] - ref[f]).max() / s < TOL_F64
        assert np.abs(m - ref).max() / s < TOL_F32
        # the paper's sufficiency criterion: |err| <= dx / (4 M) with M <= m_max on unflagged pixels
        assert np.abs(m[~f] - ref[~f]).max() <= W.dx / 4 / 3.26 if (~f).any() else True
        print(W.name, "flagged fraction", f.mean(), st)


def test_edge_cases(env):
    torch, lt, O = env
    W = workloads.make(0)
    # n_lens = 0 -> zero map in every mode
    Z = W._replace(lenses=np.zeros((0, 7)))
    for mode in (lt.LT_FP64, lt.LT_FP32, lt.LT_MIXED):
        assert np.all(_gpu_map(torch, lt, Z, mode) == 0)
    # 1 x 1, 1 x n, n x 1 grids
    for nx, ny in ((1, 1), (1, 50), (70, 1), (33, 9)):
        ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, nx, ny)
        assert _err(_gpu_map(torch, lt, W, lt.LT_FP64, nx=nx, ny=ny), ref) < TOL_F64
        m = _gpu_map(torch, lt, W, lt.LT_MIXED, nx=nx, ny=ny)
        assert np.abs(m - ref).max() / np.abs(ref).max() < TOL_F32
    # pixel exactly on a lens centre, circular lens (e = 0), more lenses than one chunk
    L = workloads.random_catalogue(77, 700, L=20.0)
    L[0, 2] = 0.0
    L[1, 2] = 0.0
    L[1, 0], L[1, 1] = 0.0, 0.0
    W2 = workloads.Workload("edge", L, -8.0, -8.0, 0.5, 40, 36, 77)      # pixel (16,16) = (0,0) = centre of lens 1
    ref = O.gradient_grid(W2.lenses, W2.x_min, W2.y_min, W2.dx, W2.nx, W2.ny)
    assert _err(_gpu_map(torch, lt, W2, lt.LT_FP64), ref) < TOL_F64
    assert _err(_gpu_map(torch, lt, W2, lt.LT_FP32), ref) < TOL_F32
    one = workloads.Workload("centre", L[1:2], 0.0, 0.0, 0.5, 1, 1, 0)
    assert np.all(_gpu_map(torch, lt, one, lt.LT_FP64) == 0)


def test_error_codes_and_bad_lens(env):
    torch, lt, O = env
    W = workloads.make(0)
    L = torch.from_numpy(W.lenses).cuda()
    with pytest.raises(lt.LtError) as e:
        lt.lt_gradient_grid(L, 0.0, 0.0, -1.0, 8, 8)
    assert e.value.code == -3
    with pytest.raises(lt.LtError) as e:
        lt.lt_gradient_grid(L, 0.0, 0.0, 1.0, 8, 8, mode=7, out=torch.empty((8, 8, 2), dtype=torch.float64, device="cuda"),
                            workspace=torch.empty(1 << 16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -4
    with pytest.raises(lt.LtError) as e:
        lt.lt_gradient_grid(L, 0.0, 0.0, 1.0, 8, 8, workspace=torch.empty(64, dtype=torch.uint8, device="cuda"))
    assert e.value.code == -5
    bad = W.lenses.copy()
    bad[3, 5] = bad[3, 4] * 0.5           # rcut < rcore
    ws = lt.alloc_workspace(len(bad), 8, 8, lt.LT_FP64)
    out = lt.lt_gradient_grid(torch.from_numpy(bad).cuda(), 0.0, 0.0, 1.0, 8, 8, workspace=ws)
    rc, k = lt.lt_last_status(ws)
    assert rc == lt.LT_ERR_BAD_LENS_PARAMS and k == 3
    assert torch.isnan(out).all()


def test_host_buffer_entry_point(env):
    torch, lt, O = env
    W = workloads.make(0)
    hL = torch.from_numpy(W.lenses).pin_memory()
    for mode, dt in ((lt.LT_FP64, torch.float64), (lt.LT_FP32, torch.float32), (lt.LT_MIXED, torch.float64)):
        hout = torch.empty((W.ny, W.nx, 2), dtype=dt).pin_memory()
        ws = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, mode, host=True)
        lt.lt_gradient_grid_host(hL, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, hout, ws)
        torch.cuda.synchronize()
        ref = _gpu_map(torch, lt, W, mode)
        assert np.array_equal(hout.numpy(), ref)
        # pageable output and the forced staging path give the same map as the kernel's direct stores into pinned memory
        pageable = torch.full((W.ny, W.nx, 2), float("nan"), dtype=dt)
        lt.lt_gradient_grid_host(hL, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, pageable, ws)
        torch.cuda.synchronize()
        assert np.array_equal(pageable.numpy(), ref)
        hout.fill_(float("nan"))
        try:
            lt.lt_set_tuning(single_launch=2)
            lt.lt_gradient_grid_host(hL, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, hout, ws)
            torch.cuda.synchronize()
        finally:
            lt.lt_set_tuning()
        assert np.array_equal(hout.numpy(), ref)


def test_row_block_sharding_stitches_to_the_unsharded_map(env):
    """DESIGN.md section 9 on one GPU: the row blocks two ranks would compute (shard.compute_block through the real
    lt_gradient_grid; mixed with its self-computed halo row) stitched together against the unsharded map and the oracle."""
    torch, lt, O = env
    from paper_1902_03252_b200 import shard
    W = workloads.make(1, paper_regime=True, n_override=301)
    L = torch.from_numpy(W.lenses).cuda()
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    s = np.abs(ref).max()

    def compute(lenses, x_min, y_min, dx, nx, ny, mode):
        return lt.lt_gradient_grid(lenses, x_min, y_min, dx, nx, ny, mode)
    for mode, tol in ((lt.LT_FP64, TOL_F64), (lt.LT_FP32, TOL_F32), (lt.LT_MIXED, TOL_F32)):
        whole = _gpu_map(torch, lt, W, mode).astype(np.float64)
        for world in (2, 3):
            parts = []
            for rank in range(world):
                b, out = shard.compute_block(compute, L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, rank, world,
                                             mixed_mode=lt.LT_MIXED)
                assert out.shape[0] == b.j1 - b.j0
                parts.append(out.cpu().numpy().astype(np.float64))
            stitched = np.concatenate(parts, axis=0)
            assert stitched.shape == whole.shape
            assert np.abs(stitched - ref).max() / s < tol
            # blocks differ from the unsharded call by the rounding of their first row's coordinate only
            assert np.abs(stitched - whole).max() / s < (1e-13 if mode == lt.LT_FP64 else tol)


def test_calibration_tool_on_small_workloads(env):
    """paper_1902_03252_b200.calibrate (its arithmetic is lt_rule_audit's, checked bit for bit against
    oracle/calibrate_ref.py in test_gpu_audit.py): for the product's tile-centre fp32 the rule, paper constants or
    calibrated, misses no pixel that violates the paper's criterion, and the implied M_max exceeds the paper's 3.26; the
    paper's plain SP version ("identical up to the change in precision") has the larger error, largest next to the
    lens centres ((A.65) P:876-880, Fig. 9) -- what the centre patches of P:284 are for."""
    torch, lt, O = env
    from paper_1902_03252_b200 import calibrate
    for W, model, mixed in ((workloads.make(1, paper_regime=True, n_override=400), "dpie", None),
                            (workloads.make_sie("small", n_override=300), "sie", (3.26, 0.0104 / 0.03, 6.0, 0.3, 1.0))):
        r = calibrate.calibrate(W, model, mixed)
        tc, pl = r["tile_centre"], r["plain"]
        assert tc["criterion"]["violating_and_missed_by_rule"] == 0
        assert tc["calibrated_rule"]["violating_and_missed"] == 0
        assert tc["calibrated_rule"]["flagged_fraction"] <= tc["criterion"]["flagged_fraction"] + 1e-12
        assert tc["implied_m_max_no_patches"] > 3.26
        # cored dPIE: both versions carry the rounding of the sum and differ by a few per cent either way (DESIGN.md
        # section 13); the singular SIE is where the plain version's coordinate rounding shows
        assert pl["sp_error_arcsec"]["max"] >= (1.0 if model == "sie" else 0.8) * tc["sp_error_arcsec"]["max"]
        if model == "sie":                                     # the paper's own case: SIS direction theta / R at the centres
            near = list(pl["max_sp_error_by_distance_px"].values())
            assert max(near[:3]) > 3 * max(near[5:])           # plain SP: worst within a few pixels of a centre
            flat = list(tc["max_sp_error_by_distance_px"].values())
            assert max(flat[:3]) < 3 * max(flat[5:])           # tile-centre coordinates: no growth towards the centres
        print(W.name, "plain", pl["sp_error_arcsec"], pl["max_sp_error_by_distance_px"])
        print(W.name, "tile centre", tc["sp_error_arcsec"], tc["max_sp_error_by_distance_px"])


def test_plain_sp_variant(env):
    """lt_set_tuning bit 4: the paper's own SP version (all of Alg. 1 l.3-14 in fp32).  Against the long-double oracle:
    <= 1e-5 of max|alpha| outside the rule's DP patches (R10), reported inside; the mixed mode run on top of it still
    delivers fp64 bits on the flagged pixels; the tuning bit leaves the fp64 mode untouched."""
    torch, lt, O = env
    W = workloads.make(1, n_override=333)._replace(ny=211)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    s = np.abs(ref).reshape(-1, 2).max(axis=0)
    g64 = _gpu_map(torch, lt, W, lt.LT_FP64)
    tile = _gpu_map(torch, lt, W, lt.LT_FP32)
    lt.lt_set_tuning(single_launch=16)
    try:
        plain = _gpu_map(torch, lt, W, lt.LT_FP32)
        ws = []
        m = _gpu_map(torch, lt, W, lt.LT_MIXED, ws_out=ws)
        flags = lt.lt_mixed_last_flags(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy()
        sp = lt.lt_mixed_last_sp_map(ws[0], len(W.lenses), W.nx, W.ny).cpu().numpy()
        assert np.array_equal(_gpu_map(torch, lt, W, lt.LT_FP64), g64)
    finally:
        lt.lt_set_tuning()
    assert np.array_equal(sp, plain) and not np.array_equal(plain, tile)
    patch = (flags & 1) != 0
    e = np.abs(plain.astype(np.float64) - ref) / s
    print("plain SP: max err outside patches %.3e, inside %.3e; tile-centre fp32 %.3e" % (
        e[~patch].max(), e[patch].max() if patch.any() else 0.0, (np.abs(tile.astype(np.float64) - ref) / s).max()))
    assert e[~patch].max() < TOL_F32
    f = flags != 0
    assert np.array_equal(m[f], g64[f]) and np.array_equal(m[~f], plain[~f].astype(np.float64))
    assert np.array_equal(flags, O.mixed_flags(sp, W.lenses, W.x_min, W.y_min, W.dx))


@pytest.mark.parametrize("name,emax,ratio,tol", [("e<=0.6, rcut/rcore 1.01-10", 0.6, (1.01, 10.0), 1e-12),
                                                  ("e<=0.9", 0.9, (1.5, 1000.0), 1e-12),
                                                  ("e<=0.99", 0.99, (1.5, 1000.0), 1e-12),
                                                  ("rcut/rcore 1.0001-1.01", 0.6, (1.0001, 1.01), 1e-10)])
def test_fp64_kernel_beyond_the_configs(env, name, emax, ratio, tol):
    """Single lenses far outside the configs' parameter ranges (strong ellipticity, rcut close to rcore, rcore down to
    1e-4", points from 1e-6" to 300" from the centre, a third of them on the lens axes) against the __float128 oracle
    (no reflection).  Everything within 1e-12 except rcut/rcore -> 1, where the scale rcut/(rcut - rcore) amplifies the
    rounding of psi_t - psi_c (outside every config; bound stated here)."""
    torch, lt, O = env
    rng = np.random.default_rng(5)
    n = 8
    L = np.empty((n, 7))
    L[:, 0], L[:, 1] = rng.uniform(-100, 100, n), rng.uniform(-100, 100, n)
    L[:, 2], L[:, 3] = rng.uniform(0, emax, n), rng.uniform(0, np.pi, n)
    L[:, 4] = np.exp(rng.uniform(np.log(1e-4), np.log(10.0), n))
    L[:, 5] = L[:, 4] * np.exp(rng.uniform(np.log(ratio[0]), np.log(ratio[1]), n))
    L[:, 6] = rng.uniform(1, 10, n)
    worst = 0.0
    for k in range(n):
        m = 4000
        r = np.exp(rng.uniform(np.log(1e-6), np.log(300.0), m))
        a = rng.uniform(0, 2 * np.pi, m)
        a = np.where(rng.integers(0, 3, m) == 0, L[k, 3] + rng.integers(0, 4, m) * np.pi / 2, a)
        px, py = L[k, 0] + r * np.cos(a), L[k, 1] + r * np.sin(a)
        ref = O.gradient_points(L[k:k + 1], px, py, O.QUAD, reflect=False)
        g = lt.lt_gradient_points(torch.from_numpy(L[k:k + 1]).cuda(),
                                  torch.from_numpy(np.stack([px, py], 1)).cuda()).cpu().numpy()
        assert np.isfinite(g).all()
        worst = max(worst, np.abs(g - ref).max() / np.abs(ref).max())
    print(name, "worst fp64 error / max|alpha|", worst)
    assert worst < tol


def test_call_is_capturable_in_a_cuda_graph(env):
    """The hot path enqueues only kernels and memsets on the caller's stream (no allocation, no synchronisation), so an
    MCMC loop can capture it once in a CUDA graph and replay it with new catalogue contents in the same buffers."""
    torch, lt, O = env
    W = workloads.make(0)
    L = torch.from_numpy(W.lenses).cuda()
    for mode, dt in ((lt.LT_FP64, torch.float64), (lt.LT_MIXED, torch.float64)):
        ws = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, mode)
        out = torch.empty((W.ny, W.nx, 2), dtype=dt, device="cuda")
        lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, out=out, workspace=ws)   # warm-up (opt-ins)
        torch.cuda.synchronize()
        expect = out.clone()
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            with torch.cuda.graph(g, stream=s):
                lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, out=out, workspace=ws, stream=s)
        out.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, expect)
        # new parameters in the same device buffer: the replay follows them
        L2 = W.lenses.copy()
        L2[:, 6] *= 2.0
        L.copy_(torch.from_numpy(L2).cuda())
        g.replay()
        torch.cuda.synchronize()
        if mode == lt.LT_FP64:
            assert torch.allclose(out, 2.0 * expect, rtol=1e-13, atol=0)
        L.copy_(torch.from_numpy(W.lenses).cuda())


@pytest.mark.parametrize("n_lens,chunk", [(1, 0), (7, 0), (9, 5), (33, 0), (64, 7)])
def test_fp32_lens_groups_and_remainders(env, n_lens, chunk):
    """The packed fp32 kernels take several lenses per iteration (dPIE 2, SIE 8) plus a lens-by-lens rest, per shared-memory
    chunk: catalogue sizes and chunk lengths (lt_set_tuning) that leave every remainder, against the oracles (1e-5), and the
    same bits whatever the chunking."""
    torch, lt, O = env
    from oracle import lt_oracle_sie as S
    nx, ny = 300, 41
    Wd = workloads.Workload("grp", workloads.random_catalogue(900 + n_lens, n_lens, L=40.0), -40.0, -6.0, 0.27, nx, ny, 0)
    rng = np.random.default_rng(950 + n_lens)
    Ls = np.stack([rng.uniform(-40, 40, n_lens), rng.uniform(-6, 6, n_lens), rng.uniform(0.0, 0.15, n_lens),
                   rng.uniform(0.0, np.pi, n_lens), rng.uniform(0.5, 3.0, n_lens)], axis=1)
    refd = O.gradient_grid(Wd.lenses, Wd.x_min, Wd.y_min, Wd.dx, nx, ny)
    refs = S.gradient_grid(Ls, Wd.x_min, Wd.y_min, Wd.dx, nx, ny)
    base = None
    for ch in sorted({0, chunk}):
        try:
            lt.lt_set_tuning(chunk32=ch)
            d = _gpu_map(torch, lt, Wd, lt.LT_FP32)
            s = lt.lt_gradient_grid_sie(torch.from_numpy(Ls).cuda(), Wd.x_min, Wd.y_min, Wd.dx, nx, ny, lt.LT_FP32)
            torch.cuda.synchronize()
            s = s.cpu().numpy()
        finally:
            lt.lt_set_tuning()
        assert _err(d, refd) < TOL_F32 and _err(s, refs) < TOL_F32, (n_lens, ch, _err(d, refd), _err(s, refs))
        if base is None:
            base = (d, s)
        else:
            assert np.array_equal(d, base[0]) and np.array_equal(s, base[1])
