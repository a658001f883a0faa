"""lt_rule_audit (the paper's accuracy criterion |err_i| <= dx / (4 M_i), eq. 24-26, evaluated on the
device) against oracle/calibrate_ref.py, bit for bit: the violation map, the counts, the error maxima and the
error-by-distance table.  First on ORACLE-made maps (the oracle's long-double map as DP map, the same map rounded to fp32
and perturbed with seeded noise as SP map, the oracle's rule as mask), then on the maps of an end-to-end LT_MIXED call."""
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
    from oracle import lt_oracle as O, calibrate_ref as C
    lt.lib()
    return torch, lt, O, C


def _compare(torch, lt, C, sp, dp, W, flags):
    centres = np.ascontiguousarray(W.lenses[:, [0, 1, 6]])
    d_res, viol = lt.lt_rule_audit(torch.from_numpy(sp).cuda(), torch.from_numpy(dp).cuda(), W.x_min, W.y_min, W.dx,
                                   centres=torch.from_numpy(centres).cuda() if len(centres) else None,
                                   flags=torch.from_numpy(flags).cuda() if flags is not None else None, want_violation=True)
    got = lt.lt_rule_audit_result(d_res, W.dx)
    expect_v = C.violations(sp, dp, W.dx)
    assert np.array_equal(viol.cpu().numpy(), expect_v)
    ref = C.audit(sp, dp, W.dx, flags)
    for k, v in ref.items():
        assert got[k] == v, (k, got[k], v)                     # integers and fp64 maxima alike: exact
    table = C.max_err_by_distance(sp, dp, centres[:, :2], W.x_min, W.y_min, W.dx)
    assert got["max_err_by_distance"] == table
    assert got["implied_m_max"] == C.implied_m_max(ref["max_err"], W.dx)
    return got


@pytest.mark.parametrize("cfg,kw,nx,ny", [(0, {}, 64, 64), (1, {"paper_regime": True, "n_override": 400}, 400, 400),
                                          (1, {"n_override": 333}, 333, 77), (0, {}, 1, 40), (0, {}, 50, 1)])
def test_audit_on_oracle_made_maps(env, cfg, kw, nx, ny):
    torch, lt, O, C = env
    W = workloads.make(cfg, **kw)._replace(nx=nx, ny=ny)
    dp = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    rng = np.random.default_rng(500 + cfg + nx)
    noise = rng.normal(0.0, W.dx / 6.0, dp.shape) * (rng.random(dp.shape) < 0.05)      # 5 % of the values off by ~dx/6
    sp = np.ascontiguousarray((dp + noise).astype(np.float32))
    flags = O.mixed_flags(sp, W.lenses, W.x_min, W.y_min, W.dx)
    got = _compare(torch, lt, C, sp, dp, W, flags)
    if W.nx * W.ny > 1000:
        assert 0 < got["n_violating"] < W.nx * W.ny
    _compare(torch, lt, C, sp, dp, W, None)                    # without a mask: everything counts as outside / missed


def test_audit_of_an_end_to_end_mixed_call(env):
    """the maps the CUDA path itself produced (config 1, paper regime, 400 x 400): the audit of lt_rule_audit equals the
    oracle's evaluation of the same three arrays; the paper's rule misses no violating pixel there"""
    torch, lt, O, C = env
    W = workloads.make(1, paper_regime=True, n_override=400)
    L = torch.from_numpy(W.lenses).cuda()
    ws = lt.alloc_workspace(len(W.lenses), W.nx, W.ny, lt.LT_MIXED)
    lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, lt.LT_MIXED, workspace=ws)
    sp = lt.lt_mixed_last_sp_map(ws, len(W.lenses), W.nx, W.ny).cpu().numpy()
    flags = lt.lt_mixed_last_flags(ws, len(W.lenses), W.nx, W.ny).cpu().numpy()
    dp = lt.lt_gradient_grid(L, W.x_min, W.y_min, W.dx, W.nx, W.ny, lt.LT_FP64).cpu().numpy()
    got = _compare(torch, lt, C, sp, dp, W, flags)
    assert got["n_violating_missed"] == 0
    print("audit", {k: got[k] for k in ("n_violating", "n_flagged", "max_err", "implied_m_max")})
