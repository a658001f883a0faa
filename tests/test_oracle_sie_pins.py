"""Pins of the SIE oracle (oracle/lt_oracle_sie.cpp = the paper's Algorithm 1) to what the paper and the
mathematics fix -- not to itself.  CPU only."""
import numpy as np

from oracle import lt_oracle_sie as S
from paper_1902_03252_b200 import workloads


def _rot(a):
    return np.array([[np.cos(a), -np.sin(a)], [np.sin(a), np.cos(a)]])


def test_sis_limit_has_constant_modulus_b0():
    """eps = 0: the SIE reduces to the SIS, whose deflection has |alpha| = theta_E = b0 everywhere (eq. 10)
    and points radially away from the centre, whatever Phi."""
    L = np.array([[1.5, -2.0, 0.0, 0.7, 3.25]])
    rng = np.random.default_rng(0)
    px, py = rng.uniform(-50, 50, 200), rng.uniform(-50, 50, 200)
    a = S.gradient_points(L, px, py)
    assert np.abs(np.hypot(a[:, 0], a[:, 1]) - 3.25).max() < 1e-15 * 3.25 * 4
    r = np.stack([px - 1.5, py + 2.0], axis=1)
    cross = a[:, 0] * r[:, 1] - a[:, 1] * r[:, 0]
    assert np.abs(cross).max() < 1e-13 and (np.sum(a * r, axis=1) > 0).all()


def test_eq21_worked_values():
    """eq. 21 by hand for Phi = 0, centre at the origin, eps = 0.2, b0 = 2 at (3, 4):
    R^2 = 0.8*9 + 1.2*16 = 26.4; grad_1 = 0.8*2*3/sqrt(26.4) = 4.8/sqrt(26.4); grad_2 = 1.2*2*4/sqrt(26.4) = 9.6/sqrt(26.4).
    Decimal values typed from a hand calculation (sqrt(26.4) = 5.138093031466052)."""
    a = S.gradient_points(np.array([[0.0, 0.0, 0.2, 0.0, 2.0]]), [3.0], [4.0])[0]
    assert abs(a[0] - 0.934198732993828) < 1e-14 and abs(a[1] - 1.868397465987655) < 1e-14
    # Phi = pi/2 swaps the roles of the axes (major axis along theta_2): the same numbers at (-4, 3) rotated by 90 degrees
    b = S.gradient_points(np.array([[0.0, 0.0, 0.2, np.pi / 2, 2.0]]), [-4.0], [3.0])[0]
    assert abs(b[0] + 1.868397465987655) < 1e-14 and abs(b[1] - 0.934198732993828) < 1e-14


def test_gradient_of_the_potential_by_finite_differences():
    """alpha = grad psi (eq. 2) with Psi_eps = b0 R (eq. 9-10 with eq. 19): 4th-order central differences of the
    potential against the oracle's gradient, many lenses, points away from the centres."""
    W = workloads.make_sie("small")
    L = W.lenses
    rng = np.random.default_rng(5)
    px, py = rng.uniform(-90, 90, 400), rng.uniform(-90, 90, 400)
    d = np.min(np.hypot(px[:, None] - L[None, :, 0], py[:, None] - L[None, :, 1]), axis=1)
    px, py = px[d > 1.0], py[d > 1.0]
    h = 1e-2

    def psi(ox, oy):
        return S.potential_points(L, px + ox, py + oy)
    g1 = (-psi(2 * h, 0) + 8 * psi(h, 0) - 8 * psi(-h, 0) + psi(-2 * h, 0)) / (12 * h)
    g2 = (-psi(0, 2 * h) + 8 * psi(0, h) - 8 * psi(0, -h) + psi(0, -2 * h)) / (12 * h)
    a = S.gradient_points(L, px, py)
    s = np.abs(a).max()
    assert np.abs(a[:, 0] - g1).max() / s < 2e-10 and np.abs(a[:, 1] - g2).max() / s < 2e-10


def test_rotation_superposition_homogeneity():
    rng = np.random.default_rng(9)
    L = np.array([[0.4, -1.1, 0.12, 0.3, 2.0]])
    px, py = rng.uniform(-30, 30, 100), rng.uniform(-30, 30, 100)
    a = S.gradient_points(L, px, py)
    # rotating the lens angle and the pixel about the centre by the same angle rotates alpha (Alg. 1 l.5-6, 10-11)
    ang = 0.77
    Rm = _rot(ang)
    q = (np.stack([px - 0.4, py + 1.1], axis=1) @ Rm.T) + np.array([0.4, -1.1])
    L2 = L.copy(); L2[0, 3] += ang
    b = S.gradient_points(L2, q[:, 0], q[:, 1])
    assert np.abs(b - a @ Rm.T).max() < 1e-14
    # Phi -> Phi + pi: same lens
    L3 = L.copy(); L3[0, 3] += np.pi
    assert np.abs(S.gradient_points(L3, px, py) - a).max() < 1e-14
    # degree-0 homogeneity about the centre: alpha(c + t r) = alpha(c + r) (eq. 21: theta / R)
    b = S.gradient_points(L, 0.4 + 7.5 * (px - 0.4), -1.1 + 7.5 * (py + 1.1))
    assert np.abs(b - a).max() < 1e-13
    # superposition (eq. 14-15) and linearity in b0
    W = workloads.make_sie("small")
    tot = S.gradient_points(W.lenses, px, py)
    parts = sum(S.gradient_points(W.lenses[k:k + 1], px, py) for k in range(len(W.lenses)))
    assert np.abs(tot - parts).max() / np.abs(tot).max() < 1e-14
    L4 = L.copy(); L4[0, 4] *= 3.0
    assert np.abs(S.gradient_points(L4, px, py) - 3.0 * a).max() < 1e-14


def test_centre_pixel_and_grid_layout():
    L = np.array([[1.0, 2.0, 0.1, 0.4, 5.0]])
    assert np.all(S.gradient_points(L, [1.0], [2.0]) == 0)          # reading R5: R = 0 contributes nothing
    W = workloads.make_sie("small")
    g = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, 7, 5)
    i, j = np.meshgrid(np.arange(7), np.arange(5))
    p = S.gradient_points(W.lenses, W.x_min + i.ravel() * W.dx, W.y_min + j.ravel() * W.dx)
    assert np.array_equal(g.reshape(-1, 2), p)                      # [ny, nx, 2], x fastest
    s = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, 7, 5, row_stride=2)
    assert np.array_equal(s[::2], g[::2]) and np.isnan(s[1::2]).all()
    # the DP and SP versions are "identical up to the change in precision"
    d = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, 7, 5, precision=S.DOUBLE)
    f = S.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, 7, 5, precision=S.FLOAT)
    m = np.abs(g).max()
    assert np.abs(d - g).max() / m < 1e-14 and 1e-9 < np.abs(f - g).max() / m < 1e-4


def test_benchmark_catalogue_matches_the_papers_description():
    """Section 4: 6730 x 6730 px at 0.03", 2 + 700 halos; b0 from eq. 22 with sigma_v = 1000 / 700 km/s and
    10-15 km/s: 4 pi (1000/299792.458)^2 rad = 28.84", (700): 14.13", galaxies 2.9e-3 .. 6.5e-3 arcsec."""
    W = workloads.make_sie("paper")
    assert W.nx == W.ny == 6730 and abs(W.dx - 0.03) < 1e-15 and len(W.lenses) == 702
    assert abs(W.lenses[0, 4] - 28.84) < 0.005 and abs(W.lenses[1, 4] - 14.13) < 0.005
    assert W.lenses[0, 2] == 0.05 and W.lenses[1, 2] == 0.04
    g = W.lenses[2:]
    assert g[:, 4].min() > 2.88e-3 and g[:, 4].max() < 6.5e-3 and g[:, 2].min() >= 0 and g[:, 2].max() <= 0.15
    assert W.nx * W.ny * len(W.lenses) == 31795615800           # 3.18e10 interactions
