"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code involved).

Each test is chosen so that a plausible mistake in oracle/lt_oracle.cpp (dropped term, wrong sign, swapped rotation,
conjugated log, wrong prefactor) fails at least one:
  golden / Form Q      : definition alpha = grad psi via the surface-density quadrature (eq. 2-4)
  div/curl             : laplace psi = 2 kappa, curl grad = 0 (eq. 2-3)
  far field / slope    : monopole |alpha| R -> (1-e^2) b0 rcut, central slope b0 R / (2 rcore)
  symmetries           : Algorithm 1's rotations, superposition (eq. 14-15)
  mixed rule           : the constants the paper prints
"""
import numpy as np
import mpmath as mp
import pytest

from oracle import lt_oracle as O
from oracle import form_q
from paper_1902_03252_b200 import workloads

mp.mp.dps = 30


def _rel(a, b):
    return float(abs(a - b) / max(abs(b), mp.mpf(10) ** -30))


def test_golden_long_double_and_double(golden):
    _, cases = golden
    for rows, t1, t2, g1, g2 in cases:
        scale = max(abs(g1), abs(g2))
        # Form C carries an absolute rounding error ~ b0/(2 sqrt(e)) * eps_T per lens (prefactor times a log near 0):
        # for L3 (e = 1e-6) at the pixel 0.002" from its centre that is 1.6e-15 relative in long double and 7e-12 in
        # double -- the reason the reference is the long double instantiation (reading R7).
        for prec, tol in ((O.LONG_DOUBLE, 5e-15), (O.DOUBLE, 2e-11), (O.QUAD, 3e-16)):
            v = O.gradient_points(rows, [t1], [t2], prec)[0]
            assert abs(mp.mpf(float(v[0])) - g1) / scale < tol, (rows, t1, t2, prec)
            assert abs(mp.mpf(float(v[1])) - g2) / scale < tol, (rows, t1, t2, prec)


def test_form_q_random_tiny():
    """Form C (C++) == quadrature of the density at random points of random lenses, incl. e up to 0.6,
    points close to the centre and close to the removable 0/0 point (0, +2 w sqrt(e)) of Form C."""
    rng = np.random.default_rng(7)
    for trial in range(12):
        e = [0.6, 0.45, 0.1, 1e-3, 1e-6, 0.3][trial % 6]
        lens = (rng.uniform(-3, 3), rng.uniform(-3, 3), e, rng.uniform(0, np.pi), rng.uniform(0.05, 1.0),
                rng.uniform(5, 50), rng.uniform(1, 10))
        c, s = np.cos(lens[3]), np.sin(lens[3])
        pts = [(lens[0] + rng.uniform(-20, 20), lens[1] + rng.uniform(-20, 20)),
               (lens[0] + 1e-3 * rng.uniform(-1, 1), lens[1] + 1e-3 * rng.uniform(-1, 1))]
        for w in (lens[4], lens[5]):            # near the focus point, lens frame (0, 2 w sqrt(e)) -> sky frame
            yf = 2 * w * np.sqrt(e) * (1 + 1e-7)
            pts.append((lens[0] - yf * s + 1e-7, lens[1] + yf * c))
        for (t1, t2) in pts:
            g1, g2 = form_q.gradient_point([lens], t1, t2)
            v = O.gradient_points([lens], [t1], [t2], O.LONG_DOUBLE)[0]
            # relative 1e-14 plus Form C's absolute floor ~ b0/(2 sqrt(e)) eps_longdouble (see the golden test)
            tol = 1e-14 * max(abs(g1), abs(g2)) + 16 * lens[6] / (2 * np.sqrt(e)) * 1.1e-19
            assert abs(mp.mpf(float(v[0])) - g1) < tol, (lens, t1, t2)
            assert abs(mp.mpf(float(v[1])) - g2) < tol, (lens, t1, t2)


@pytest.mark.parametrize("e,rcore,rcut", [(0.9, 0.3, 12.0), (0.95, 0.5, 30.0), (0.99, 0.2, 8.0), (0.3, 1.0, 1.01),
                                          (0.6, 2.0, 2.0002), (0.9, 1.0, 1.001)])
def test_form_q_beyond_the_configs(e, rcore, rcut):
    """Outside every config (e >= 0.9, rcut/rcore -> 1): the __float128 instantiation, which the GPU test
    test_fp64_kernel_beyond_the_configs compares with, equals the density quadrature to the rounding of its fp64
    output; the long double one loses rcut/(rcut - rcore) times its rounding in the difference of the two PIEMD terms."""
    lens = (0.7, -0.4, e, 0.8, rcore, rcut, 5.0)
    amp = rcut / (rcut - rcore)
    for (t1, t2) in [(3.1, 2.2), (0.75, -0.38), (-14.0, 9.0), (0.7 + 1e-3, -0.4 - 2e-3)]:
        g1, g2 = form_q.gradient_point([lens], t1, t2)
        s = max(abs(g1), abs(g2))
        q = O.gradient_points([lens], [t1], [t2], O.QUAD)[0]
        qn = O.gradient_points([lens], [t1], [t2], O.QUAD, reflect=False)[0]      # as the GPU test calls it
        v = O.gradient_points([lens], [t1], [t2], O.LONG_DOUBLE)[0]
        for k, g in ((0, g1), (1, g2)):
            assert abs(mp.mpf(float(q[k])) - g) / s < 3e-16, (lens, t1, t2, k)
            assert abs(mp.mpf(float(qn[k])) - g) / s < 3e-16, (lens, t1, t2, k)
            # long double: relative rounding plus Form C's absolute floor ~ b0/(2 sqrt(e)) eps (see the golden test),
            # both amplified by rcut/(rcut - rcore)
            tol = 3e-16 * s + amp * 1.1e-19 * (64 * s + 16 * lens[6] / (2 * np.sqrt(e)))
            assert abs(mp.mpf(float(v[k])) - g) < tol, (lens, t1, t2, k)


def test_reflection_evaluation_matches_unreflected_and_quad():
    """Reading R21: evaluating Form C at (x,-|y|) changes nothing (away from the 0/0 point)."""
    W = workloads.make(0)
    rng = np.random.default_rng(3)
    px, py = rng.uniform(-50, 50, 500), rng.uniform(-50, 50, 500)
    a = O.gradient_points(W.lenses, px, py, O.LONG_DOUBLE, reflect=True)
    b = O.gradient_points(W.lenses, px, py, O.LONG_DOUBLE, reflect=False)
    q = O.gradient_points(W.lenses, px, py, O.QUAD, reflect=False)
    s = np.abs(q).max()
    assert np.abs(a - b).max() / s < 1e-15
    assert np.abs(a - q).max() / s < 1e-15


def test_elliptical_form_tends_to_circular_closed_form():
    """e -> 0 of Form C meets the north star's closed form linearly in e (connects the two oracle branches)."""
    base = np.array([[0.3, -0.2, 0.0, 0.7, 0.4, 25.0, 3.0]])
    px, py = np.array([2.0, -7.0, 0.31, 40.0]), np.array([1.0, 3.0, -0.19, -35.0])
    circ = O.gradient_points(base, px, py)
    prev = None
    for e in (1e-4, 1e-6, 1e-8):
        L = base.copy(); L[0, 2] = e
        d = np.abs(O.gradient_points(L, px, py) - circ).max() / np.abs(circ).max()
        assert d < 3 * e
        if prev is not None:
            assert d < prev / 30          # linear convergence
        prev = d


def test_circular_closed_form_central_slope_and_far_field():
    b0, rc, rt = 3.0, 0.4, 25.0
    L = np.array([[0.0, 0.0, 0.0, 0.0, rc, rt, b0]])
    # central slope b0 R / (2 rcore) (relative correction -(R/rcore)^2 (1 + rcore/rcut + ...)/4 ~ 2e-8 at R = 1e-4)
    v = O.gradient_points(L, [1e-4], [0.0])[0]
    assert abs(v[0] / (b0 * 1e-4 / (2 * rc)) - 1) < 1e-7 and v[1] == 0
    # pixel exactly on the centre: zero (reading R5), elliptical too
    assert np.all(O.gradient_points(L, [0.0], [0.0]) == 0)
    L2 = L.copy(); L2[0, 2] = 0.3
    assert np.abs(O.gradient_points(L2, [0.0], [0.0])).max() < 1e-18
    # far field: |alpha| R -> (1 - e^2) b0 rcut (total mass pi b0 rcut (1-e^2) of the density in the header)
    for e in (0.0, 0.3, 0.6):
        L3 = L.copy(); L3[0, 2] = e; L3[0, 3] = 0.9
        R = 1e8
        v = O.gradient_points(L3, [R * 0.6], [R * 0.8])[0]
        assert abs(np.hypot(*v) * R / ((1 - e * e) * b0 * rt) - 1) < 1e-6
        assert abs(v[0] / v[1] - 0.75) < 1e-6      # radial


def test_circular_closed_form_small_radius_series():
    """Reading R22: for R << rcore the closed form has the series b0 R/(2 rcore) - b0 s R^3/8 (1/rcore^3 - 1/rcut^3) + O(R^5),
    s = rcut/(rcut-rcore) (from sqrt(w^2+R^2) - w = R^2/2w - R^4/8w^3 + ...).  The literal difference of square roots
    loses ulp(rcut)/R there (1e-6 relative at R = 1e-5, rcut = 1000 even in long double); the oracle's rearranged
    evaluation must meet the series to fp64 rounding."""
    b0, rc, rt = 7.0, 0.4, 1000.0
    L = np.array([[0.0, 0.0, 0.0, 0.0, rc, rt, b0]])
    for R in (1e-5, 1e-4, 1e-3):
        v = O.gradient_points(L, [R * 0.6], [-R * 0.8])[0]
        series = b0 * R / (2 * rc) - b0 * rt / (rt - rc) * R ** 3 / 8 * (1 / rc ** 3 - 1 / rt ** 3)
        assert abs(np.hypot(*v) / series - 1) < 5e-16 + (R / rc) ** 4
        assert abs(v[0] / v[1] + 0.75) < 1e-15
        q = O.gradient_points(L, [R * 0.6], [-R * 0.8], O.QUAD)[0]
        assert np.abs(v - q).max() / np.abs(q).max() < 3e-16


def test_div_is_2kappa_and_curl_is_zero():
    """4th-order central differences of the oracle's own alpha: div = 2 kappa (elementary expression), curl = 0."""
    W = workloads.make(0)
    rng = np.random.default_rng(11)
    px, py = rng.uniform(-45, 45, 300), rng.uniform(-45, 45, 300)
    # keep away from lens centres by > 0.5" so that the 5th derivative stays tame
    d = np.min(np.hypot(px[:, None] - W.lenses[None, :, 0], py[:, None] - W.lenses[None, :, 1]), axis=1)
    px, py = px[d > 0.5], py[d > 0.5]
    h = 2e-3

    def A(ox, oy):
        return O.gradient_points(W.lenses, px + ox, py + oy)
    def d_dx(c):
        return (-A(2 * h, 0)[:, c] + 8 * A(h, 0)[:, c] - 8 * A(-h, 0)[:, c] + A(-2 * h, 0)[:, c]) / (12 * h)
    def d_dy(c):
        return (-A(0, 2 * h)[:, c] + 8 * A(0, h)[:, c] - 8 * A(0, -h)[:, c] + A(0, -2 * h)[:, c]) / (12 * h)
    kappa = O.kappa_points(W.lenses, px, py)
    div = d_dx(0) + d_dy(1)
    curl = d_dy(0) - d_dx(1)
    assert np.abs(div - 2 * kappa).max() < 1e-8 * max(1.0, np.abs(kappa).max())
    assert np.abs(curl).max() < 1e-8 * max(1.0, np.abs(kappa).max())


def test_superposition_and_linearity():
    W = workloads.make(0)
    rng = np.random.default_rng(5)
    px, py = rng.uniform(-50, 50, 200), rng.uniform(-50, 50, 200)
    total = O.gradient_points(W.lenses, px, py)
    parts = sum(O.gradient_points(W.lenses[k:k + 1], px, py) for k in range(len(W.lenses)))
    assert np.abs(total - parts).max() / np.abs(total).max() < 1e-15
    L2 = W.lenses.copy(); L2[:, 6] *= 2.5
    assert np.abs(O.gradient_points(L2, px, py) - 2.5 * total).max() / np.abs(total).max() < 1e-15
    # order of lenses: rounding-level only (reading R8)
    assert np.abs(O.gradient_points(W.lenses[::-1], px, py) - total).max() / np.abs(total).max() < 1e-15
    # n_lens = 0 -> zeros
    assert np.all(O.gradient_grid(np.zeros((0, 7)), -1, -1, 0.5, 4, 3) == 0)


def test_rotation_translation_reflection_symmetries():
    lens = np.array([[1.2, -0.7, 0.35, 0.4, 0.3, 18.0, 5.0]])
    rng = np.random.default_rng(9)
    px, py = rng.uniform(-10, 10, 100), rng.uniform(-10, 10, 100)
    a = O.gradient_points(lens, px, py)
    s = np.abs(a).max()
    # Phi -> Phi + pi: same lens
    l2 = lens.copy(); l2[0, 3] += np.pi
    assert np.abs(O.gradient_points(l2, px, py) - a).max() / s < 1e-14
    # rotate lens angle and pixels about the lens centre by t: alpha rotates by t
    t = 0.83
    c, sn = np.cos(t), np.sin(t)
    qx = lens[0, 0] + c * (px - lens[0, 0]) - sn * (py - lens[0, 1])
    qy = lens[0, 1] + sn * (px - lens[0, 0]) + c * (py - lens[0, 1])
    l3 = lens.copy(); l3[0, 3] += t
    b = O.gradient_points(l3, qx, qy)
    assert np.abs(b[:, 0] - (c * a[:, 0] - sn * a[:, 1])).max() / s < 1e-14
    assert np.abs(b[:, 1] - (sn * a[:, 0] + c * a[:, 1])).max() / s < 1e-14
    # translation
    l4 = lens.copy(); l4[0, 0] += 3.25; l4[0, 1] -= 1.5
    assert np.abs(O.gradient_points(l4, px + 3.25, py - 1.5) - a).max() / s < 1e-14
    # mirror about the major axis (Phi = 0 lens): alpha_y odd, alpha_x even in y
    l5 = np.array([[0.0, 0.0, 0.35, 0.0, 0.3, 18.0, 5.0]])
    u, v = O.gradient_points(l5, px, py), O.gradient_points(l5, px, -py)
    assert np.abs(u[:, 0] - v[:, 0]).max() / s < 1e-15 and np.abs(u[:, 1] + v[:, 1]).max() / s < 1e-15
    # major axis along theta_1 for Phi = 0: the mass is more extended along x, so at equal distance the
    # deflection on the minor axis is larger than on the major axis
    ax = O.gradient_points(l5, [5.0], [0.0])[0, 0]
    ay = O.gradient_points(l5, [0.0], [5.0])[0, 1]
    assert ay > ax > 0
    # CCW rotation sense (reading R2): with Phi = +pi/2 the major axis lies along theta_2
    l6 = l5.copy(); l6[0, 3] = np.pi / 2
    assert abs(O.gradient_points(l6, [0.0], [5.0])[0, 1] - ax) / ax < 1e-14
    l7 = l5.copy(); l7[0, 3] = 0.3        # small CCW tilt: point on the tilted major axis gets a purely radial pull
    p = 5.0 * np.array([np.cos(0.3), np.sin(0.3)])
    g = O.gradient_points(l7, [p[0]], [p[1]])[0]
    assert abs(g[0] * p[1] - g[1] * p[0]) < 1e-13 and abs(np.hypot(*g) - ax) / ax < 1e-14


def test_grid_matches_points_and_row_stride():
    W = workloads.make(0)
    g = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    jj, ii = np.meshgrid(np.arange(W.ny), np.arange(W.nx), indexing="ij")
    p = O.gradient_points(W.lenses, W.x_min + ii.ravel() * W.dx, W.y_min + jj.ravel() * W.dx)
    assert np.array_equal(g.reshape(-1, 2), p)
    gs = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, row_stride=4)
    assert np.array_equal(gs[::4], g[::4]) and np.all(np.isnan(gs[1::4]))
    # output layout: index 2*(j*nx+i)+c, x fastest: a lens far to the +x side pulls along +x
    assert g.shape == (W.ny, W.nx, 2)


def test_double_and_float_instantiations_are_close():
    W = workloads.make(0)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, O.LONG_DOUBLE)
    s = np.abs(ref).max()
    assert np.abs(O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, O.DOUBLE) - ref).max() / s < 1e-12
    assert np.abs(O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny, O.FLOAT) - ref).max() / s < 1e-3


def test_quad_audit_of_long_double_on_stress_sample():
    """__float128 (unreflected) audit of the long-double reference on config-4-like inputs: pixels nearest the
    centres, near-circular lenses.  Records the oracle's own error (must be far below the 1e-12 parity gate)."""
    W = workloads.make(4)
    L = W.lenses[:40]
    rng = np.random.default_rng(2)
    k = rng.integers(0, len(L), 300)
    i = np.round((L[k, 0] - W.x_min) / W.dx) + rng.integers(-1, 2, 300)
    j = np.round((L[k, 1] - W.y_min) / W.dx) + rng.integers(-1, 2, 300)
    px, py = W.x_min + i * W.dx, W.y_min + j * W.dx
    a = O.gradient_points(L, px, py, O.LONG_DOUBLE)
    q = O.gradient_points(L, px, py, O.QUAD, reflect=False)
    err = np.abs(a - q).max() / np.abs(q).max()
    assert err < 2e-14, err


# ------------------------------------------------------------------ mixed rule (section 3.2-3.3)

def test_printed_constants_of_the_rule():
    assert abs(0.03 / 4 - 7.5e-3) < 1e-15
    assert round(7.5e-3 / 2.3e-3, 2) == 3.26
    assert round(0.03 / 3.26, 4) == 0.0092
    assert 2 * 400 ** 2 + 700 * 20 ** 2 == 600000              # P:930 (approx 1 % of 6730^2)
    assert abs(600000 / 6730 ** 2 - 0.01) < 0.004


def _linear_map(nx, ny, dx, a, b, c, d):
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    t1, t2 = ii * dx, jj * dx
    return np.stack([a * t1 + b * t2, c * t1 + d * t2], axis=-1).astype(np.float32)


@pytest.mark.parametrize("a,b,c,d,expect", [
    (0.0, 0.0, 0.0, 0.0, 0),            # no lensing: M = 1
    (0.5, 0.0, 0.0, 0.0, 0),            # M_1 = 2 <= 3.26
    (0.75, 0.0, 0.0, 0.0, 2),           # |dx - 0.75 dx| = 0.0075 < 0.0092  -> eq. 25 on delta_1
    (0.0, 0.0, 0.0, 1.25, 2),           # parity flip, |dx - 1.25 dx| = 0.0075   -> eq. 25 on delta_2
    (1.7, 0.0, 0.0, 0.0, 0),            # |dx - 1.7 dx| = 0.021 > 0.0092
    (0.0, 0.3, 0.0, 0.0, 0),            # |delta_3| = 0.009 < 0.0104
    (0.0, 0.4, 0.0, 0.0, 4),            # |delta_3| = 0.012 > 0.0104      -> eq. 28
    (0.0, 0.0, -0.4, 0.0, 4),           # |delta_4| = 0.012               -> eq. 28
    (0.8, 0.0, 0.5, 0.0, 6),
])
def test_rule_at_the_papers_pixel_scale(a, b, c, d, expect):
    """At dx = 0.03" the scaled thresholds are the paper's printed 0.0092" (eq. 25) and 0.0104" (eq. 28)."""
    dx = 0.03
    sp = _linear_map(9, 7, dx, a, b, c, d)
    far = np.array([[1e6, 1e6, 0.1, 0.0, 0.1, 10.0, 1.0]])       # patch off-grid
    flags = O.mixed_flags(sp, far, 0.0, 0.0, dx)
    assert np.all(flags == expect), flags


def test_rule_axis_of_extent_one_and_patches():
    dx = 0.03
    sp = _linear_map(9, 1, dx, 0.75, 0.4, 0.0, 0.0)
    far = np.array([[1e6, 1e6, 0.1, 0.0, 0.1, 10.0, 1.0]])
    assert np.all(O.mixed_flags(sp, far, 0.0, 0.0, dx) == 2)      # ny = 1: delta_2, delta_3 skipped (R12)
    # patches at the paper's scale: 400x400 / 20x20 px become (2*200+1)^2 / (2*10+1)^2 boxes (R14)
    L = np.array([[15.0, 15.0, 0.1, 0.0, 5.0, 500.0, 25.0], [3.0, 27.0, 0.1, 0.0, 0.1, 10.0, 1.0]])
    sp = np.zeros((1000, 1000, 2), np.float32)
    f = O.mixed_flags(sp, L, 0.0, 0.0, dx)
    assert (f == 1).sum() == 401 * 401 + 21 * 21 and set(np.unique(f)) == {0, 1}
    assert f[500, 500] == 1 and f[900, 100] == 1 and f[900, 111] == 0 and f[500, 701] == 0
    # clipped at the edge
    L2 = np.array([[0.0, 0.0, 0.1, 0.0, 0.1, 10.0, 1.0]])
    assert (O.mixed_flags(sp, L2, 0.0, 0.0, dx) == 1).sum() == 11 * 11


def test_mixed_map_flagged_pixels_carry_dp_values():
    W = workloads.make(0)
    m, flags = O.mixed_map(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    ref = O.gradient_grid(W.lenses, W.x_min, W.y_min, W.dx, W.nx, W.ny)
    assert np.array_equal(m[flags != 0], ref[flags != 0])
    assert np.array_equal(m[flags == 0], ref[flags == 0].astype(np.float32).astype(np.float64))
