"""Pins of the NFW oracle (oracle/lt_oracle_nfw.cpp) to what the mathematics fixes -- not to itself.  CPU only."""
import numpy as np
from scipy import integrate

from oracle import lt_oracle_nfw as N
from paper_1902_03252_b200 import workloads


def test_deflection_is_the_enclosed_mass_of_the_convergence():
    """Circular lens: alpha(R) = (2/R) int_0^R kappa(r) r dr (eq. 2-3 P:60-62 for a circular kappa), with kappa the
    elementary NFW convergence, by adaptive quadrature -- an independent route to the deflection."""
    ks, rs = 0.23, 37.0
    L = np.array([[0.0, 0.0, 0.0, 0.0, ks, rs]])
    for R in (0.02, 1.0, 11.0, 36.9, 37.0, 37.5, 120.0, 900.0):
        m, _ = integrate.quad(lambda r: N.kappa(r, ks, rs) * r, 0.0, R, points=[rs] if R > rs else None,
                              epsabs=0, epsrel=1e-13, limit=400)
        a = N.gradient_points(L, [R], [0.0])[0]
        assert abs(a[0] / (2.0 * m / R) - 1) < 5e-12 and a[1] == 0


def test_values_at_the_scale_radius_and_limits():
    ks, rs = 0.31, 12.5
    L = np.array([[1.0, -2.0, 0.0, 0.4, ks, rs]])
    # x = 1: F = 1, alpha = 4 ks rs (1 - ln 2); continuity across x = 1
    a = N.gradient_points(L, [1.0 + rs], [-2.0])[0]
    assert abs(a[0] - 4 * ks * rs * (1 - np.log(2.0))) < 1e-14 * 4 * ks * rs
    lo = N.gradient_points(L, [1.0 + rs * (1 - 1e-9)], [-2.0])[0][0]
    hi = N.gradient_points(L, [1.0 + rs * (1 + 1e-9)], [-2.0])[0][0]
    assert abs(lo - a[0]) < 1e-7 and abs(hi - a[0]) < 1e-7
    # x -> 0: alpha -> 4 ks rs * (x/2) (ln(2/x) - 1/2); x -> infinity: alpha -> 4 ks rs (ln(x/2) + pi/(2x)) / x
    x = 1e-4
    a = N.gradient_points(L, [1.0 + rs * x], [-2.0])[0][0]
    assert abs(a / (4 * ks * rs * 0.5 * x * (np.log(2 / x) - 0.5)) - 1) < 1e-6
    x = 1e6
    a = N.gradient_points(L, [1.0 + rs * x], [-2.0])[0][0]
    assert abs(a / (4 * ks * rs * (np.log(x / 2) + np.pi / (2 * x)) / x) - 1) < 1e-9
    assert np.all(N.gradient_points(L, [1.0], [-2.0]) == 0)
    # the long-double values against the __float128 instantiation, down to x = 1e-5
    px = 1.0 + rs * np.array([1e-5, 1e-3, 0.3, 0.999, 1.001, 7.0])
    q = N.gradient_points(L, px, np.full(6, -2.0), N.QUAD)
    r = N.gradient_points(L, px, np.full(6, -2.0))
    assert np.abs(r - q).max() / (4 * ks * rs) < 1e-13


def test_literal_formula_in_40_digits_incl_the_neighbourhood_of_the_scale_radius():
    """Reading R27: the oracle evaluates arccosh(1/x), arccos(1/x) as atanh / atan of sqrt(|1 - x^2|).  The literal textbook
    formula, in 40-digit arithmetic (mpmath), is the reference here -- including |1 - x| down to 1e-9, where the literal
    route loses eps/|1 - x| in long double."""
    import mpmath as mp
    mp.mp.dps = 40
    ks, rs = 0.27, 41.0

    def alpha(x):
        x = mp.mpf(x)
        if x < 1:
            F = mp.acosh(1 / x) / mp.sqrt(1 - x * x)
        elif x > 1:
            F = mp.acos(1 / x) / mp.sqrt(x * x - 1)
        else:
            F = mp.mpf(1)
        return 4 * mp.mpf(ks) * rs * (mp.log(x / 2) + F) / x
    L = np.array([[0.0, 0.0, 0.0, 0.0, ks, rs]])
    for x in (1e-3, 0.2, 0.5, 1 - 1e-3, 1 - 1e-6, 1 - 1e-9, 1 + 1e-9, 1 + 1e-6, 1 + 1e-3, 3.0, 250.0):
        R = rs * x
        exact = alpha(mp.mpf(R) / rs)                    # the x the oracle sees: R / rs with R the fp64 number
        got = N.gradient_points(L, [R], [0.0])[0][0]
        assert abs(got - float(exact)) <= 4e-16 * 4 * ks * rs, x


def test_gradient_of_the_potential_by_finite_differences():
    """alpha = grad psi (eq. 2) for the pseudo-elliptical potential psi_eps(theta) = psi(R) (eq. 19)"""
    W = workloads.make_nfw()
    L = W.lenses[:12]
    rng = np.random.default_rng(2)
    px, py = rng.uniform(-90, 90, 300), rng.uniform(-90, 90, 300)
    d = np.min(np.hypot(px[:, None] - L[None, :, 0], py[:, None] - L[None, :, 1]), axis=1)
    px, py = px[d > 0.5], py[d > 0.5]
    h = 5e-3

    def psi(ox, oy):
        return N.potential_points(L, px + ox, py + oy)
    g1 = (-psi(2 * h, 0) + 8 * psi(h, 0) - 8 * psi(-h, 0) + psi(-2 * h, 0)) / (12 * h)
    g2 = (-psi(0, 2 * h) + 8 * psi(0, h) - 8 * psi(0, -h) + psi(0, -2 * h)) / (12 * h)
    a = N.gradient_points(L, px, py)
    s = np.abs(a).max()
    assert np.abs(a[:, 0] - g1).max() / s < 1e-9 and np.abs(a[:, 1] - g2).max() / s < 1e-9


def test_symmetries():
    rng = np.random.default_rng(3)
    L = np.array([[0.4, -1.1, 0.15, 0.3, 0.2, 9.0]])
    px, py = rng.uniform(-30, 30, 100), rng.uniform(-30, 30, 100)
    a = N.gradient_points(L, px, py)
    ang = 0.77
    Rm = np.array([[np.cos(ang), -np.sin(ang)], [np.sin(ang), np.cos(ang)]])
    q = (np.stack([px - 0.4, py + 1.1], axis=1) @ Rm.T) + np.array([0.4, -1.1])
    L2 = L.copy(); L2[0, 3] += ang
    assert np.abs(N.gradient_points(L2, q[:, 0], q[:, 1]) - a @ Rm.T).max() < 1e-13
    L3 = L.copy(); L3[0, 3] += np.pi
    assert np.abs(N.gradient_points(L3, px, py) - a).max() < 1e-13
    L4 = L.copy(); L4[0, 4] *= 3.0                       # linear in kappa_s
    assert np.abs(N.gradient_points(L4, px, py) - 3.0 * a).max() < 1e-13
    W = workloads.make_nfw()
    tot = N.gradient_points(W.lenses, px, py)
    parts = sum(N.gradient_points(W.lenses[k:k + 1], px, py) for k in range(len(W.lenses)))
    assert np.abs(tot - parts).max() / np.abs(tot).max() < 1e-14
    g = N.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, 6, 4)
    i, j = np.meshgrid(np.arange(6), np.arange(4))
    assert np.array_equal(g.reshape(-1, 2), N.gradient_points(W.lenses, W.x_min + i.ravel() * W.dx, W.y_min + j.ravel() * W.dx))
