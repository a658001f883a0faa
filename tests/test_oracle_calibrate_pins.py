"""Pins of oracle/calibrate_ref.py (the paper's accuracy criterion, eq. 24-26) against what the
paper prints and against hand-made maps on which every quantity is known in closed form.  CPU only."""
import numpy as np
import pytest

from oracle import calibrate_ref as C

DX = 0.03          # the paper's pixel size


def linear_map(a, b, nx, ny, dx=DX, c=0.0, d=0.0):
    """grad = (a x + c y, b y + d x) on the grid x = i dx, y = j dx: delta_1 = a dx, delta_2 = b dx everywhere"""
    x = np.arange(nx) * dx
    y = np.arange(ny) * dx
    g = np.empty((ny, nx, 2))
    g[..., 0] = a * x[None, :] + c * y[:, None]
    g[..., 1] = b * y[:, None] + d * x[None, :]
    return g


def test_printed_constants():
    # P:280 a quarter of a pixel; P:284 7.5e-3 / 2.3e-3 = 3.26; P:303 / P:312: M_i > 3.26 <=> |dx - delta| < 0.0092"
    assert DX / 4 == pytest.approx(7.5e-3, rel=1e-12)
    assert C.implied_m_max(2.3e-3, DX) == pytest.approx(3.26, abs=5e-3)
    assert DX / 3.26 == pytest.approx(0.0092, abs=5e-5)


def test_magnification_of_linear_maps_incl_edges_and_parity_flip():
    # a != b so that a swap of the components or of the axes shows; a > 1: image parity flips, |.| matters
    for a, b in ((0.25, 0.5), (1.5, -0.75), (0.0, 0.9)):
        g = linear_map(a, b, 7, 5, c=0.3, d=-0.2)        # the cross terms must not enter delta_1, delta_2
        M1, M2 = C.magnifications(g, DX)
        assert np.allclose(M1, 1.0 / abs(1.0 - a), rtol=1e-9) and np.allclose(M2, 1.0 / abs(1.0 - b), rtol=1e-9)
        # first column / first row use the forward neighbour (R12): same value on a linear map, and finite
        assert np.isfinite(M1[:, 0]).all() and np.isfinite(M2[0, :]).all()


def test_edge_rule_is_the_forward_neighbour():
    g = np.zeros((3, 4, 2))
    g[:, :, 0] = np.array([0.0, 1.0, 3.0, 6.0])[None, :] * DX          # delta_1: column 0 -> g[1]-g[0], then backward
    g[:, :, 1] = np.array([0.0, 2.0, 3.0])[:, None] * DX
    d1, d2 = C.axis_deltas(g)
    assert np.allclose(d1[0], np.array([1.0, 1.0, 2.0, 3.0]) * DX) and np.allclose(d2[:, 0], np.array([2.0, 2.0, 1.0]) * DX)
    # an axis of extent 1 has no neighbour: delta = 0, M = 1
    M1, M2 = C.magnifications(g[:1], DX)
    assert np.all(M2 == 1.0) and M1.shape == (1, 4)


def test_violation_threshold_is_the_papers_budget():
    # M_1 = 3.26 exactly on axis 1 (|dx - delta_1| = dx / 3.26 = 0.0092"), M_2 = 1: budgets 2.3e-3" and 7.5e-3"
    a = 1.0 - 1.0 / 3.26
    dp = linear_map(a, 0.0, 6, 4)
    budget1, budget2 = DX / 4 / 3.26, DX / 4
    assert budget1 == pytest.approx(2.3e-3, abs=5e-6)
    for e1, e2, expect in ((0.99 * budget1, 0.0, 0), (1.01 * budget1, 0.0, 1), (0.0, 0.99 * budget2, 0),
                           (0.0, 1.01 * budget2, 2), (1.01 * budget1, 1.01 * budget2, 3),
                           (0.0, 1.01 * budget1, 0)):        # an error of axis 2 is not judged by the budget of axis 1
        sp = dp.copy()
        sp[2, 3, 0] += e1
        sp[2, 3, 1] -= e2
        v = C.violations(sp, dp, DX)
        assert v[2, 3] == expect and v.sum() == expect


def test_audit_counts_against_a_mask():
    dp = linear_map(0.5, 0.5, 8, 8)
    sp = dp.astype(np.float32).astype(np.float64)
    sp[1, 1, 0] += 1.0          # violating, flagged
    sp[5, 6, 1] += 1.0          # violating, missed
    flags = np.zeros((8, 8), np.uint8)
    flags[1, 1] = 2
    flags[0, 0] = 1             # a patch pixel
    r = C.audit(sp, dp, DX, flags)
    assert (r["n_violating"], r["n_violating_flagged"], r["n_violating_missed"], r["n_flagged"]) == (2, 1, 1, 2)
    assert r["max_err"] == pytest.approx(1.0, rel=1e-6) and r["max_err_in_patch"] < 1e-6 and r["n_pixels"] == 64
    assert C.implied_m_max(r["max_err"], DX) == pytest.approx(DX / 4, rel=1e-6)


def test_max_err_by_distance_bins():
    nx = ny = 300
    dp = np.zeros((ny, nx, 2))
    sp = np.zeros((ny, nx, 2))
    # one centre exactly on pixel (150, 150); errors planted at Chebyshev distances 0, 1, 3, 130
    for (i, j, e) in ((150, 150, 5.0), (151, 150, 4.0), (150, 147, 3.0), (20, 150, 2.0)):
        sp[j, i, 1] = e
    got = C.max_err_by_distance(sp, dp, [(150 * DX, 150 * DX)], 0.0, 0.0, DX)
    assert got == [5.0, 4.0, 3.0, 0.0, 0.0, 0.0, 0.0, 0.0, 2.0]
    # a second centre next to the far pixel moves it into the first bin (nearest centre counts)
    got = C.max_err_by_distance(sp, dp, [(150 * DX, 150 * DX), (20.2 * DX, 150.1 * DX)], 0.0, 0.0, DX)
    assert got[0] == 5.0 and got[8] == 0.0
