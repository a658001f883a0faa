"""Properties of the CUDA path that hold at any size, for the three lens models (tier 3): superposition
over lenses (eq. 14-15), permutation of the catalogue, translation of grid and lenses together, a quarter
turn of the whole configuration: the maps are compared with each other.  And the short-list kernel of
lt_gradient_points (one warp per point) against the oracle, the grid kernel and the thread-per-point kernel."""
import numpy as np
import pytest

from paper_1902_03252_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    from paper_1902_03252_b200 import lt
    lt.lib()
    return torch, lt


def _models(lt):
    return {"dpie": (lt.lt_gradient_grid, workloads.make(1, paper_regime=True, n_override=160), 3),
            "sie": (lt.lt_gradient_grid_sie, workloads.make_sie("small", n_override=160), 3),
            "nfw": (lt.lt_gradient_grid_nfw, workloads.make_nfw(n_override=160), 3)}


def _map(torch, fn, lenses, W, mode=0, x_min=None, y_min=None, nx=None, ny=None):
    L = torch.from_numpy(np.ascontiguousarray(lenses)).cuda()
    out = fn(L, W.x_min if x_min is None else x_min, W.y_min if y_min is None else y_min, W.dx,
             W.nx if nx is None else nx, W.ny if ny is None else ny, mode)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("model", ["dpie", "sie", "nfw"])
def test_superposition_and_permutation(env, model):
    torch, lt = env
    fn, W, angle_col = _models(lt)[model]
    n = len(W.lenses)
    whole = _map(torch, fn, W.lenses, W)
    s = np.abs(whole).max()
    parts = _map(torch, fn, W.lenses[: n // 3], W) + _map(torch, fn, W.lenses[n // 3:], W)
    assert np.abs(whole - parts).max() / s < 1e-14
    perm = np.random.default_rng(1).permutation(n)
    assert np.abs(_map(torch, fn, W.lenses[perm], W) - whole).max() / s < 1e-14
    # fp32: the same up to single precision rounding
    w32 = _map(torch, fn, W.lenses, W, mode=1)
    assert np.abs(_map(torch, fn, W.lenses[perm], W, mode=1) - w32).max() / s < 5e-6
    # an empty catalogue gives exactly zero, a doubled catalogue exactly twice the map's worth of terms
    assert np.all(_map(torch, fn, W.lenses[:0], W) == 0)
    assert np.abs(_map(torch, fn, np.concatenate([W.lenses, W.lenses]), W) - 2 * whole).max() / s < 1e-14


@pytest.mark.parametrize("model", ["dpie", "sie", "nfw"])
def test_translation_and_quarter_turn(env, model):
    torch, lt = env
    fn, W, angle_col = _models(lt)[model]
    whole = _map(torch, fn, W.lenses, W)
    s = np.abs(whole).max()
    # shift grid and lenses by the same vector: theta - theta_center changes only by the rounding of the shifted numbers
    sh = np.array([37.25, -18.5])
    Ls = W.lenses.copy()
    Ls[:, 0] += sh[0]; Ls[:, 1] += sh[1]
    shifted = _map(torch, fn, Ls, W, x_min=W.x_min + sh[0], y_min=W.y_min + sh[1])
    assert np.abs(shifted - whole).max() / s < 1e-12
    # quarter turn about the origin: (x, y) -> (-y, x), Phi -> Phi + pi/2; the deflection turns with it
    Lr = W.lenses.copy()
    Lr[:, 0], Lr[:, 1] = -W.lenses[:, 1], W.lenses[:, 0]
    Lr[:, angle_col] = W.lenses[:, angle_col] + np.pi / 2
    # rotated grid: new pixel (i', j') sits at (x', y') = (-y_j, x_i): i' runs over -y (descending j), j' over x
    xs = W.x_min + np.arange(W.nx) * W.dx
    ys = W.y_min + np.arange(W.ny) * W.dx
    rot = _map(torch, fn, Lr, W, x_min=-ys[-1], y_min=xs[0], nx=W.ny, ny=W.nx)
    # rot[j', i'] with x' = -ys[-1] + i' dx = -y_j  ->  j = ny-1-i';  y' = xs[0] + j' dx = x_i  ->  i = j'
    back = np.empty_like(whole)
    back[..., 0] = rot[:, ::-1, 1].T          # alpha_x(x, y) =  alpha'_y(x', y')
    back[..., 1] = -rot[:, ::-1, 0].T         # alpha_y(x, y) = -alpha'_x(x', y')
    assert np.abs(back - whole).max() / s < 1e-12


@pytest.mark.parametrize("model", ["dpie", "sie", "nfw"])
def test_short_point_lists(env, model):
    """lt_gradient_points up to 4096 points: one warp per point, lenses dealt to the lanes.  Against the oracle (1e-12),
    against the thread-per-point kernel and the grid map (same terms, another order of the sum), independent of the
    length of the list, for catalogue sizes around the lane count (ragged last round, fewer lenses than lanes, none)."""
    torch, lt = env
    fn, W, _ = _models(lt)[model]
    if model == "dpie":
        from oracle import lt_oracle as Om
        pts_fn = lt.lt_gradient_points
    elif model == "sie":
        from oracle import lt_oracle_sie as Om
        pts_fn = lt.lt_gradient_points_sie
    else:
        from oracle import lt_oracle_nfw as Om
        pts_fn = lt.lt_gradient_points_nfw
    rng = np.random.default_rng(8)
    i, j = rng.integers(0, W.nx, 333), rng.integers(0, W.ny, 333)
    px, py = W.x_min + i * W.dx, W.y_min + j * W.dx
    pts = torch.from_numpy(np.stack([px, py], axis=1)).cuda()
    for n in (len(W.lenses), 65, 64, 33, 31, 1, 0):
        lenses = np.ascontiguousarray(W.lenses[:n])
        L = torch.from_numpy(lenses).cuda()
        short = pts_fn(L, pts).cpu().numpy()
        if n == 0:
            assert np.all(short == 0)
            continue
        ref = Om.gradient_points(lenses, px, py)
        s = np.abs(ref).max()
        assert np.abs(short - ref).max() / s < 1e-12
        try:
            lt.lt_set_tuning(single_launch=4)
            per_thread = pts_fn(L, pts).cpu().numpy()
        finally:
            lt.lt_set_tuning()
        grid = _map(torch, fn, lenses, W)[j, i]
        assert np.array_equal(per_thread, grid)
        assert np.abs(short - grid).max() / s < 4e-15
        assert np.array_equal(pts_fn(L, pts[:100].contiguous()).cpu().numpy(), short[:100])
        assert np.array_equal(pts_fn(L, pts[:1].contiguous()).cpu().numpy(), short[:1])


def test_two_host_threads_two_streams(env):
    """The library keeps no per-call state outside the caller's workspace (launch counts and event hooks are per host
    thread, the occupancy cache is locked): two host threads driving different models and modes on their own streams at
    the same time get the bits of the serial runs."""
    import threading
    torch, lt = env
    jobs = [(lt.lt_gradient_grid, workloads.make(1, paper_regime=True, n_override=300), lt.LT_MIXED),
            (lt.lt_gradient_grid_sie, workloads.make_sie("small", n_override=280), lt.LT_FP64),
            (lt.lt_gradient_grid_nfw, workloads.make_nfw(n_override=260), lt.LT_FP32),
            (lt.lt_gradient_grid, workloads.make(1, paper_regime=True, n_override=240), lt.LT_FP64)]
    serial = [_map(torch, fn, W.lenses, W, mode) for fn, W, mode in jobs]
    results, errors = [None] * len(jobs), []

    def work(k):
        try:
            fn, W, mode = jobs[k]
            st = torch.cuda.Stream()
            L = torch.from_numpy(np.ascontiguousarray(W.lenses)).cuda()
            torch.cuda.synchronize()
            with torch.cuda.stream(st):
                for _ in range(25):
                    out = fn(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, mode, stream=st)
                    n_launch = lt.lt_last_launch_count()
                    assert n_launch >= 2
            st.synchronize()
            results[k] = out.cpu().numpy().astype(np.float64)
        except Exception as e:  # noqa: BLE001 -- reported by the main thread
            errors.append((k, repr(e)))
    threads = [threading.Thread(target=work, args=(k,)) for k in range(len(jobs))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    for k in range(len(jobs)):
        assert np.array_equal(results[k], serial[k]), k


@pytest.mark.parametrize("model", ["dpie", "sie", "nfw"])
def test_dependent_launch_does_not_change_the_result(env, model):
    """The grid, patch, flag and list kernels are launched as programmatic dependents of the kernel before them and wait
    for it before they read anything; with the attribute switched off (lt_set_tuning, bit 3 of
    single_launch) every mode gives the same bits."""
    torch, lt = env
    fn, W, _ = _models(lt)[model]
    for mode in (0, 1, 2):
        with_pdl = [_map(torch, fn, W.lenses, W, mode) for _ in range(3)]
        try:
            lt.lt_set_tuning(single_launch=8)
            without = _map(torch, fn, W.lenses, W, mode)
        finally:
            lt.lt_set_tuning()
        for m in with_pdl:
            assert np.array_equal(m, without), (model, mode)
