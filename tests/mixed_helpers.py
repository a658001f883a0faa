"""Shared checks of the mixed-precision mask (reading R18).  No oracle input comes from the CUDA path:
  * rule_parity: the rule kernels (lt_mixed_rule) and the oracle's rule on the SAME oracle-made single precision map
    (the oracle's reference map rounded to fp32) -- bit-exact;
  * mask_agrees_away_from_thresholds: the mask the end-to-end LT_MIXED call produced on its own fp32 map against the
    oracle's mask on the oracle's map, on every pixel whose four criterion values are not within `margin` of a threshold
    (there the two fp32 maps, which differ at rounding level, may decide differently: several results are correct)."""
import numpy as np


def rule_parity(torch, lt, O, ref_map, rule_catalogue, W, mixed):
    sp = np.ascontiguousarray(ref_map.astype(np.float32))
    expect = O.mixed_flags(sp, rule_catalogue, W.x_min, W.y_min, W.dx, mixed=mixed)
    centres = torch.from_numpy(np.ascontiguousarray(rule_catalogue[:, [0, 1, 6]])).cuda()
    flags, ws = lt.lt_mixed_rule(torch.from_numpy(sp).cuda(), W.x_min, W.y_min, W.dx, centres, mixed=mixed)
    torch.cuda.synchronize()
    got = flags.cpu().numpy()
    assert np.array_equal(got, expect)
    st = lt.lt_mixed_last_stats(ws)
    assert st["n_flagged"] == int((expect != 0).sum()) and st["n_patch"] == int((expect & 1).astype(bool).sum())
    assert st["n_eq25"] == int((expect & 2).astype(bool).sum()) and st["n_eq28"] == int((expect & 4).astype(bool).sum())
    return expect


def mask_agrees_away_from_thresholds(O, flags_gpu, ref_map, rule_catalogue, W, mixed, margin_rel=1e-2, max_excluded=0.2):
    sp = np.ascontiguousarray(ref_map.astype(np.float32))
    expect, crit = O.mixed_flags(sp, rule_catalogue, W.x_min, W.y_min, W.dx, mixed=mixed, want_crit=True)
    t25, t28, m = W.dx / mixed[0], mixed[1] * W.dx, margin_rel * W.dx
    near = (np.abs(crit[..., 0] - t25) < m) | (np.abs(crit[..., 1] - t25) < m) | \
           (np.abs(crit[..., 2] - t28) < m) | (np.abs(crit[..., 3] - t28) < m)
    assert near.mean() <= max_excluded, near.mean()
    assert np.array_equal(flags_gpu[~near], expect[~near])
    assert np.array_equal(flags_gpu & 1, expect & 1)                # the patch bit does not depend on the map at all
    return near.mean()
