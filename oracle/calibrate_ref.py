"""CPU oracle of the paper's accuracy criterion (section 3.2; eq. 24-26).  TEST INFRASTRUCTURE, NOT
THE PRODUCT: only tests/ may import this module; it imports nothing from paper_1902_03252_b200 and shares no code with
the CUDA path (whose counterpart is lt_rule_audit).  Plain numpy, fp64, every step in the order the paper states it.

What the paper says:
  * "the value of grad Psi can be considered accurate enough if the error E is smaller than a quarter of a pixel"
    (P:280): E_i <= dx / 4 = 7.5e-3" at dx = 0.03".
  * "The resulting error budget ... becomes thus E_i <= 7.5e-3 arcsec / M_i, where M_i is the magnification along the
    theta_i-axis".
  * delta_1(t1, t2) = grad_1(t1, t2) - grad_1(t1 - dx, t2), delta_2(t1, t2) = grad_2(t1, t2) - grad_2(t1, t2 - dx)
    (eq. 24); the pixel length in the source plane along axis i is |dx - delta_i| (eq. 26), hence
    M_i = dx / |dx - delta_i| and the budget of component i is dx / (4 M_i) = |dx - delta_i| / 4.
  * with an SP error bound E_SP the rule's constant is M_max = (dx / 4) / E_SP (7.5e-3 / 2.3e-3 = 3.26).
Readings: R12 -- at i = 0 (j = 0) the forward neighbour stands in for the missing backward one; an axis of
extent 1 has no neighbour, its delta is taken as 0 (M_i = 1: the unmagnified budget dx / 4); R13 -- D_LS/D_OS = 1.
The magnifications are those of the DP map (the SP map is the one under test).

A pixel VIOLATES the criterion when |SP_i - DP_i| > |dx - delta_i| / 4 for i = 1 or i = 2 (bit 0: axis 1, bit 1: axis 2).
Arithmetic, so that a device implementation can be compared bit for bit: every operation below is one correctly rounded
fp64 operation (SP values widened exactly), the factor 1/4 is an exact scaling.
"""
import numpy as np


def axis_deltas(dp_map):
    """delta_1, delta_2 of eq. 24 on a [ny, nx, 2] fp64 map, backward differences, forward at the first column / row
    (R12), zero along an axis of extent 1."""
    g = np.asarray(dp_map, dtype=np.float64)
    ny, nx = g.shape[0], g.shape[1]
    d1 = np.zeros((ny, nx))
    d2 = np.zeros((ny, nx))
    if nx > 1:
        d1[:, 1:] = g[:, 1:, 0] - g[:, :-1, 0]          # grad_1(t1, t2) - grad_1(t1 - dx, t2)
        d1[:, 0] = g[:, 1, 0] - g[:, 0, 0]              # i = 0: forward neighbour
    if ny > 1:
        d2[1:, :] = g[1:, :, 1] - g[:-1, :, 1]          # grad_2(t1, t2) - grad_2(t1, t2 - dx)
        d2[0, :] = g[1, :, 1] - g[0, :, 1]              # j = 0: forward neighbour
    return d1, d2


def source_pixel_lengths(dp_map, dx):
    """|dx - delta_i| (eq. 26): the length of the pixel along axis i after lensing into the source plane."""
    d1, d2 = axis_deltas(dp_map)
    return np.abs(dx - d1), np.abs(dx - d2)


def magnifications(dp_map, dx):
    """M_i = dx / |dx - delta_i| (eq. 26); inf on a critical line."""
    s1, s2 = source_pixel_lengths(dp_map, dx)
    with np.errstate(divide="ignore"):
        return dx / s1, dx / s2


def violations(sp_map, dp_map, dx):
    """uint8 [ny, nx]: bit 0 set where |SP_1 - DP_1| > dx / (4 M_1), bit 1 where |SP_2 - DP_2| > dx / (4 M_2)."""
    sp = np.asarray(sp_map).astype(np.float64)
    dp = np.asarray(dp_map, dtype=np.float64)
    s1, s2 = source_pixel_lengths(dp, dx)
    e1 = np.abs(sp[..., 0] - dp[..., 0])
    e2 = np.abs(sp[..., 1] - dp[..., 1])
    return ((e1 > 0.25 * s1).astype(np.uint8) | ((e2 > 0.25 * s2).astype(np.uint8) << 1))


def implied_m_max(e_sp, dx):
    """M_max = (dx / 4) / E_SP  (7.5e-3 / 2.3e-3 = 3.26)."""
    return dx / 4.0 / e_sp


def audit(sp_map, dp_map, dx, flags=None):
    """Counts and error maxima of an SP map against a DP map: what lt_rule_audit returns.  flags: the rule's mask
    (bit 0 = DP centre patch), optional."""
    sp = np.asarray(sp_map).astype(np.float64)
    dp = np.asarray(dp_map, dtype=np.float64)
    v = violations(sp, dp, dx) != 0
    err = np.maximum(np.abs(sp[..., 0] - dp[..., 0]), np.abs(sp[..., 1] - dp[..., 1]))     # arcsec, worse component
    out = {"n_pixels": int(v.size), "n_violating": int(v.sum()), "max_err": float(err.max())}
    if flags is not None:
        f = np.asarray(flags)
        fl, patch = f != 0, (f & 1) != 0
        out.update({"n_flagged": int(fl.sum()), "n_violating_flagged": int((v & fl).sum()),
                    "n_violating_missed": int((v & ~fl).sum()),
                    "max_err_in_patch": float(err[patch].max()) if patch.any() else 0.0,
                    "max_err_outside_patch": float(err[~patch].max()) if (~patch).any() else 0.0})
    return out


DISTANCE_EDGES = (0.0, 1.0, 2.0, 4.0, 8.0, 16.0, 32.0, 64.0, 128.0)      # pixels; the last bin is open


def max_err_by_distance(sp_map, dp_map, centres_xy, x_min, y_min, dx):
    """Largest |SP - DP| (worse component, arcsec) among the pixels whose Chebyshev distance (in pixels) to the NEAREST
    lens centre falls in [edge_k, edge_k+1): the analogue of the paper's Fig. 9 as a table.  Brute force: the
    distance map is the minimum over all lenses.  Empty bins hold 0."""
    sp = np.asarray(sp_map).astype(np.float64)
    dp = np.asarray(dp_map, dtype=np.float64)
    ny, nx = dp.shape[0], dp.shape[1]
    err = np.maximum(np.abs(sp[..., 0] - dp[..., 0]), np.abs(sp[..., 1] - dp[..., 1]))
    best = np.full((ny, nx), np.inf)
    ii = np.arange(nx, dtype=np.float64)[None, :]
    jj = np.arange(ny, dtype=np.float64)[:, None]
    for xc, yc in np.asarray(centres_xy, dtype=np.float64).reshape(-1, 2):
        a, b = (xc - x_min) / dx, (yc - y_min) / dx                 # centre in pixel units
        best = np.minimum(best, np.maximum(np.abs(ii - a), np.abs(jj - b)))
    out = []
    edges = list(DISTANCE_EDGES) + [np.inf]
    for lo, hi in zip(edges[:-1], edges[1:]):
        m = (best >= lo) & ((best < hi) | np.isinf(hi))            # no centre at all: distance inf, last bin
        out.append(float(err[m].max()) if m.any() else 0.0)
    return out
