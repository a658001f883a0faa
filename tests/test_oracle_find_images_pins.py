"""Pins of oracle/find_images.py (the triangle search of the paper's section 2.2.2, Fig. 1) to what the
mathematics fixes.  CPU only."""
import numpy as np

from oracle import find_images as F
from oracle import lt_oracle as O


def test_no_lens_every_point_is_its_own_image():
    """gradPsi = 0: beta = theta (eq. 13), so a source strictly inside a triangle is found exactly once, in the triangle
    that contains it geometrically, at its own position; a source on the cut diagonal is reported by both triangles of
    the cell, a source on a node by the six triangles that share the node (closed triangles, reading R24)."""
    nx, ny, dx, x0, y0 = 9, 7, 0.5, -2.0, -1.0
    g = np.zeros((ny, nx, 2))
    rng = np.random.default_rng(1)
    src = np.stack([rng.uniform(x0, x0 + (nx - 1) * dx, 40), rng.uniform(y0, y0 + (ny - 1) * dx, 40)], axis=1)
    h = F.find_images(g, x0, y0, dx, 1.0, src)
    assert len(h) == 40 and np.array_equal(h["source"], np.arange(40))
    assert np.abs(h["x"] - src[:, 0]).max() < 1e-13 and np.abs(h["y"] - src[:, 1]).max() < 1e-13
    i = np.floor((src[:, 0] - x0) / dx).astype(int)
    j = np.floor((src[:, 1] - y0) / dx).astype(int)
    u, v = (src[:, 0] - x0) / dx - i, (src[:, 1] - y0) / dx - j
    assert np.array_equal(h["cell"], j * nx + i)
    assert np.array_equal(h["triangle"], (u + v > 1).astype(int))          # T0 below the diagonal u + v = 1, T1 above
    # on the diagonal of cell (2, 3): both triangles; on the interior node (4, 2): six triangles
    d = F.find_images(g, x0, y0, dx, 1.0, [[x0 + 2.5 * dx, y0 + 3.5 * dx]])
    assert [(r["cell"], r["triangle"]) for r in d] == [(3 * nx + 2, 0), (3 * nx + 2, 1)]
    n = F.find_images(g, x0, y0, dx, 1.0, [[x0 + 4 * dx, y0 + 2 * dx]])
    assert len(n) == 6 and np.abs(n["x"] - (x0 + 4 * dx)).max() < 1e-13


def _alpha_circ(R, b0, rc, rt):
    """circular dPIE deflection (north star's closed form)"""
    return b0 * rt / (rt - rc) * ((np.sqrt(rc * rc + R * R) - rc) - (np.sqrt(rt * rt + R * R) - rt)) / R


def test_cored_circular_lens_three_images_at_the_roots_of_the_lens_equation():
    """A circular cored lens and a source on the axis inside the caustic: the lens equation beta = x - alpha(|x|) sign(x)
    (eq. 1 / 13) has three roots on the axis, found here by bisection -- independent of the triangle search.  The
    search must report exactly three images, at those roots up to the linear-interpolation error of the grid."""
    b0, rc, rt = 12.0, 1.5, 400.0
    L = np.array([[0.0, 0.0, 0.0, 0.0, rc, rt, b0]])
    n, half = 241, 30.0
    dx = 2 * half / (n - 1)
    x0 = -half + 0.37 * dx                                  # no node on the axis or the centre
    g = O.gradient_grid(L, x0, x0, dx, n, n)
    beta_s = 1.3

    def f(x):
        return x - np.sign(x) * _alpha_circ(abs(x), b0, rc, rt) - beta_s
    roots = []
    for lo, hi in ((-25.0, -5.0), (-5.0, -1e-6), (5.0, 25.0)):
        assert f(lo) * f(hi) < 0
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            lo, hi = (mid, hi) if f(lo) * f(mid) > 0 else (lo, mid)
        roots.append(0.5 * (lo + hi))
    h = F.find_images(g, x0, x0, dx, 1.0, [[beta_s, 0.0]])
    assert len(h) == 3
    found = np.sort(h["x"])
    assert np.abs(found - np.sort(roots)).max() < 0.05 * dx and np.abs(h["y"]).max() < 0.05 * dx
    # D_LS/D_OS scales the deflection (eq. 13): with 0.5 the same source has the images of a lens of half the strength
    h2 = F.find_images(g, x0, x0, dx, 0.5, [[beta_s, 0.0]])
    g_half = O.gradient_grid(np.array([[0.0, 0.0, 0.0, 0.0, rc, rt, b0 / 2]]), x0, x0, dx, n, n)
    h3 = F.find_images(g_half, x0, x0, dx, 1.0, [[beta_s, 0.0]])
    assert len(h2) == len(h3) and np.array_equal(h2["cell"], h3["cell"]) and np.abs(h2["x"] - h3["x"]).max() < 1e-9


def test_translation_and_source_independence():
    """Shifting grid and sources together shifts the images; sources are searched independently of each other."""
    L = np.array([[1.0, -2.0, 0.3, 0.8, 0.8, 60.0, 6.0], [-6.0, 4.0, 0.1, 2.0, 0.3, 20.0, 2.0]])
    n, dx, x0, y0 = 101, 0.4, -20.0, -20.0
    g = O.gradient_grid(L, x0, y0, dx, n, n)
    rng = np.random.default_rng(4)
    src = rng.uniform(-3, 3, (6, 2))
    h = F.find_images(g, x0, y0, dx, 1.0, src)
    assert len(h) >= 6                                       # at least one image each (odd-number theorem: 1, 3 or 5)
    counts = np.bincount(h["source"], minlength=6)
    assert (counts % 2 == 1).all()
    for k in range(6):
        hk = F.find_images(g, x0, y0, dx, 1.0, src[k:k + 1])
        sel = h[h["source"] == k]
        assert np.array_equal(hk["cell"], sel["cell"]) and np.array_equal(hk["x"], sel["x"])
    s = 16.0                                                 # a shift that is exact in binary for these coordinates
    Ls = L.copy(); Ls[:, 0] += s; Ls[:, 1] += s
    gs = O.gradient_grid(Ls, x0 + s, y0 + s, dx, n, n)
    hs = F.find_images(gs, x0 + s, y0 + s, dx, 1.0, src + s)
    assert np.array_equal(hs["cell"], h["cell"]) and np.abs(hs["x"] - s - h["x"]).max() < 1e-9
