"""Pins of oracle/chi2.py (barycentre of the lensed-back images, eq. 11) to hand-computed values and to the closed form of
a singular isothermal sphere, through the oracle chain only.  CPU only."""
import numpy as np

from oracle import chi2 as C
from oracle import find_images as FI
from oracle import lt_oracle_sie as S


def test_hand_computed_values():
    theta = [[1.0, 2.0], [3.0, 4.0], [7.0, 7.0]]
    alpha = [[0.5, 0.5], [1.0, -1.0], [1.0, 2.0]]
    b = C.source_barycentres(theta, alpha, [0, 2, 2, 3], 2.0)      # beta = (0,1), (1,6) | none | (5,3)
    assert np.array_equal(b[0], [0.5, 3.5]) and np.isnan(b[1]).all() and np.array_equal(b[2], [5.0, 3.0])
    # system 0: observed (0,0), (3,4), predicted (0,1), (3,4), (10,10) [one of them reported twice: a shared edge];
    # system 1: one observed image, nothing predicted; system 2: observed (1,1), predicted (2,1)
    obs = [[0.0, 0.0], [3.0, 4.0], [9.0, 9.0], [1.0, 1.0]]
    sig = [0.5, 2.0, 1.0, 0.25]
    total, matched, unmatched, terms = C.chi2(obs, sig, [0, 2, 3, 4], [0, 0, 0, 0, 2], [0.0, 3.0, 3.0, 10.0, 2.0],
                                              [1.0, 4.0, 4.0, 10.0, 1.0])
    assert total == 4.0 + 0.0 + 16.0 and matched == 3 and unmatched == 1
    assert np.array_equal(terms[[0, 1, 3]], [4.0, 0.0, 16.0]) and np.isnan(terms[2])
    # a predicted image of ANOTHER system next to an observed one is not used
    total2, _, _, _ = C.chi2(obs, sig, [0, 2, 3, 4], [0, 0, 0, 2, 2], [0.0, 3.0, 10.0, 2.0, 0.0], [1.0, 4.0, 10.0, 1.0, 0.0])
    assert total2 == 4.0 + 0.0 + 16.0
    # exact dyadic translation of everything leaves chi^2 alone; sigma -> 2 sigma divides it by 4
    sh = np.array([8.0, -16.0])
    t3, _, _, _ = C.chi2(np.array(obs) + sh, sig, [0, 2, 3, 4], [0, 0, 0, 0, 2],
                         np.array([0.0, 3.0, 3.0, 10.0, 2.0]) + sh[0], np.array([1.0, 4.0, 4.0, 10.0, 1.0]) + sh[1])
    t4, _, _, _ = C.chi2(obs, 2 * np.array(sig), [0, 2, 3, 4], [0, 0, 0, 0, 2], [0.0, 3.0, 3.0, 10.0, 2.0],
                         [1.0, 4.0, 4.0, 10.0, 1.0])
    assert t3 == total and t4 == total / 4


def test_singular_isothermal_sphere_closed_form():
    """SIS with Einstein radius b0 (eq. 10): a source at beta, |beta| < b0, has the two images beta +- b0 * beta/|beta|.
    Model them with b0' = b0 + delta: the images lensed back land at beta -+ delta * beta/|beta|, their barycentre is beta
    exactly, the predicted images are beta +- b0' * beta/|beta|, each delta away from the observed one, so
    chi^2 = 2 delta^2 / sigma^2 (eq. 11)."""
    b0, delta, sigma = 2.0, 0.04, 0.1
    beta = np.array([0.36, 0.48])                                  # |beta| = 0.6
    u = beta / 0.6
    obs = np.array([beta + b0 * u, beta - b0 * u])
    model = np.array([[0.0, 0.0, 0.0, 0.0, b0 + delta]])
    alpha = S.gradient_points(model, obs[:, 0], obs[:, 1])
    bary = C.source_barycentres(obs, alpha, [0, 2], 1.0)
    assert np.abs(bary[0] - beta).max() < 1e-15
    lensed_back = obs - alpha
    assert np.abs(lensed_back[0] - (beta - delta * u)).max() < 1e-15 and np.abs(lensed_back[1] - (beta + delta * u)).max() < 1e-15
    n, dx = 321, 0.02                                              # nodes at odd multiples of dx/2: none on the centre
    x_min = -(n - 1) / 2 * dx - dx / 2
    g = S.gradient_grid(model, x_min, x_min, dx, n, n)
    hits = FI.find_images(g, x_min, x_min, dx, 1.0, bary)
    total, matched, unmatched, terms = C.chi2(obs, [sigma, sigma], [0, 2], hits["source"], hits["x"], hits["y"])
    assert matched == 2 and unmatched == 0
    assert abs(total / (2 * delta ** 2 / sigma ** 2) - 1) < 2e-3
    # the true model: chi^2 vanishes up to the interpolation error of the triangles (second order in the pixel size)
    g0 = S.gradient_grid(np.array([[0.0, 0.0, 0.0, 0.0, b0]]), x_min, x_min, dx, n, n)
    a0 = S.gradient_points(np.array([[0.0, 0.0, 0.0, 0.0, b0]]), obs[:, 0], obs[:, 1])
    h0 = FI.find_images(g0, x_min, x_min, dx, 1.0, C.source_barycentres(obs, a0, [0, 2], 1.0))
    t0, m0, _, _ = C.chi2(obs, [sigma, sigma], [0, 2], h0["source"], h0["x"], h0["y"])
    assert m0 == 2 and t0 < 2 * (0.01 * dx / sigma) ** 2          # each image within a hundredth of a pixel
