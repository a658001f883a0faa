"""Seeded synthetic lens catalogues and grids (BASELINE.json:configs; recipe in DESIGN.md section 4).

This module holds NONE of the method's arithmetic: it only draws parameters.  It is the one module both the tests of
the CPU oracle and the CUDA path take their inputs from (it imports neither).  numpy only.

A catalogue is a float64 array [n_lens, 7] with columns (xc, yc, ellipticity, angle, rcore, rcut, b0) -- arcsec and
radians -- i.e. the `lt_lens` struct of include/lt_gradient.h.  Synthetic stand-ins for the paper's HFF-like cluster
(2 cluster-scale + 700 galaxy-scale halos on an HST grid): the paper's halo positions are not published.
"""
from collections import namedtuple

import numpy as np

Workload = namedtuple("Workload", "name lenses x_min y_min dx nx ny seed")

#            name            n_pix L     n_lens seed
_CONFIGS = {
    0: ("cfg0_64x64_8", 64, 50.0, 8, 1000),
    1: ("cfg1_1024x1024_100", 1024, 100.0, 100, 1001),
    2: ("cfg2_2048x2048_500", 2048, 100.0, 500, 1002),
    3: ("cfg3_4096x4096_1000", 4096, 100.0, 1000, 1003),
    4: ("cfg4_stress_2048x2048_200", 2048, 100.0, 200, 1004),
}


def grid(n, L):
    """n x n pixel centres over [-L, L]: dx = 2L/n, first pixel at -L + dx/2 (reading R4)."""
    dx = 2.0 * L / n
    return -L + dx / 2, -L + dx / 2, dx


def _galaxies(rng, n, centre_draw):
    out = np.empty((n, 7))
    for k in range(n):                         # fixed draw order per lens: centre, e, Phi, rcore, rcut, b0
        xc, yc = centre_draw()
        out[k] = (xc, yc, rng.uniform(0.0, 0.6), rng.uniform(0.0, np.pi), rng.uniform(0.01, 1.0),
                  rng.uniform(5.0, 50.0), rng.uniform(1.0, 10.0))
    return out


def _cluster(rng):
    return np.array([rng.uniform(-5, 5), rng.uniform(-5, 5), rng.uniform(0.0, 0.6), rng.uniform(0.0, np.pi),
                     rng.uniform(5.0, 20.0), rng.uniform(500.0, 1000.0), rng.uniform(20.0, 30.0)])


def make(cfg, paper_regime=False, n_override=None, seed_offset=0):
    """Workload for BASELINE.json config `cfg` (0..4).

    paper_regime: galaxy-scale b0 x 0.05 and rcut x 0.3 (cluster halo unchanged) -- the lens-physically light variant
    on which the mixed rule flags a few percent of the pixels as in the paper's Fig. 7.
    n_override: use an n x n grid over the same extent instead (parity tests at reduced size).
    seed_offset: added to the config's seed (bench.py --gpus N: rank r draws its own catalogue with seed + r).
    """
    name, n, L, n_lens, seed = _CONFIGS[cfg]
    seed += int(seed_offset)
    rng = np.random.default_rng(seed)
    if n_override is not None:
        n = int(n_override)
        name += "_n%d" % n
    x_min, y_min, dx = grid(n, L)
    if cfg == 0:
        lenses = _galaxies(rng, n_lens, lambda: (rng.uniform(-L, L), rng.uniform(-L, L)))
    elif cfg == 1:
        cl = _cluster(rng)
        lenses = np.vstack([cl, _galaxies(rng, n_lens - 1, lambda: (rng.uniform(-L, L), rng.uniform(-L, L)))])
    elif cfg in (2, 3):
        cl = _cluster(rng)

        def gauss():
            while True:
                x, y = rng.normal(0.0, 40.0), rng.normal(0.0, 40.0)
                if abs(x) < L and abs(y) < L:
                    return x, y
        lenses = np.vstack([cl, _galaxies(rng, n_lens - 1, gauss)])
    elif cfg == 4:
        # stress: near-circular lenses, every centre within 0.05" of a pixel of the FULL 2048 grid
        x0f, y0f, dxf = grid(_CONFIGS[4][1], L)

        def near_pixel():
            while True:
                x, y = rng.normal(0.0, 40.0), rng.normal(0.0, 40.0)
                if abs(x) < L - 1 and abs(y) < L - 1:
                    break
            i, j = round((x - x0f) / dxf), round((y - y0f) / dxf)
            r, a = rng.uniform(1e-4, 0.05), rng.uniform(0.0, 2 * np.pi)
            return x0f + i * dxf + r * np.cos(a), y0f + j * dxf + r * np.sin(a)
        cl = _cluster(rng)
        cl[0], cl[1] = near_pixel()
        lenses = np.vstack([cl, _galaxies(rng, n_lens - 1, near_pixel)])
        lenses[:, 2] = 10.0 ** rng.uniform(-6.0, -3.0, size=n_lens)
    else:
        raise KeyError(cfg)
    if paper_regime:
        gal = lenses[:, 6] < 15.0
        lenses[gal, 6] *= 0.05
        lenses[gal, 5] *= 0.3
        name += "_paper_regime"
    assert np.all(lenses[:, 5] > lenses[:, 4])
    return Workload(name, np.ascontiguousarray(lenses), x_min, y_min, dx, n, n, seed)


def random_catalogue(seed, n_lens, L=50.0, e_max=0.6):
    """Generic galaxy-like catalogue for property tests."""
    rng = np.random.default_rng(seed)
    out = _galaxies(rng, n_lens, lambda: (rng.uniform(-L, L), rng.uniform(-L, L)))
    out[:, 2] *= e_max / 0.6
    return out


# ---------------------------------------------------------------------------------------------- SIE (the paper's body)
# A catalogue of SIE lenses is a float64 array [n_lens, 5]: (xc, yc, epsilon, Phi, b0) = `lt_sie_lens`.
ARCSEC_PER_RAD = 206264.80624709636
C_KM_S = 299792.458


def b0_from_sigma_v(sigma_km_s):
    """eq. 22: b0 = 4 pi (sigma_v / c)^2, converted from radians to arcsec (D_LS/D_OS = 1)."""
    return 4.0 * np.pi * (np.asarray(sigma_km_s, dtype=np.float64) / C_KM_S) ** 2 * ARCSEC_PER_RAD


def make_sie(kind="paper", n_override=None, seed_offset=0):
    """Synthetic stand-in for the paper's benchmark (section 4): 6730 x 6730 pixels at 0.03"/pixel, two
    cluster-scale SIE halos (sigma_v = 1000 and 700 km/s, epsilon = 0.05 and 0.04) and 700 galaxy-scale halos (sigma_v
    uniform in 10-15 km/s, epsilon uniform in 0-0.15).  The paper gives no positions or angles: cluster centres are
    drawn uniform in [-20,20]^2, galaxy centres Gaussian (sigma 40") redrawn until inside the grid, angles uniform in
    [0, pi).  kind = "small": 96 x 96 pixels over the same extent and 2 + 30 halos (the oracle finishes in well under
    a second).  n_override: n x n pixels over the same extent."""
    if kind == "paper":
        name, n, n_gal, seed = "sie_paper_6730x6730_702", 6730, 700, 2000
    elif kind == "small":
        name, n, n_gal, seed = "sie_small_96x96_32", 96, 30, 2001
    else:
        raise ValueError("kind must be 'paper' or 'small'")
    L = 0.5 * 6730 * 0.03
    seed += int(seed_offset)
    rng = np.random.default_rng(seed)
    if n_override is not None:
        n = int(n_override)
        name += "_n%d" % n
    x_min, y_min, dx = grid(n, L)
    out = np.empty((2 + n_gal, 5))
    for k, (sig, eps) in enumerate(((1000.0, 0.05), (700.0, 0.04))):
        out[k] = (rng.uniform(-20, 20), rng.uniform(-20, 20), eps, rng.uniform(0.0, np.pi), b0_from_sigma_v(sig))
    for k in range(n_gal):                     # fixed draw order per lens: centre, sigma_v, epsilon, Phi
        while True:
            xc, yc = rng.normal(0.0, 40.0, 2)
            if abs(xc) < L and abs(yc) < L:
                break
        sig = rng.uniform(10.0, 15.0)
        out[2 + k] = (xc, yc, rng.uniform(0.0, 0.15), rng.uniform(0.0, np.pi), b0_from_sigma_v(sig))
    return Workload(name, out, x_min, y_min, dx, n, n, seed)


# ---------------------------------------------------------------------------------------------- NFW
# A catalogue of pseudo-elliptical NFW lenses is a float64 array [n_lens, 6]: (xc, yc, epsilon, Phi, kappa_s, rs).
def make_nfw(n_override=None, seed_offset=0):
    """Synthetic cluster of NFW halos on a 512 x 512 grid over [-100, 100]": 2 cluster-scale halos (kappa_s U(0.15, 0.3),
    rs U(40, 80)", epsilon U(0, 0.2), centres U(-20, 20)^2) + 62 galaxy-scale halos (kappa_s U(0.02, 0.08), rs U(1, 5)",
    epsilon U(0, 0.2), centres N(0, 40^2) redrawn until inside), angles U(0, pi); seed 3000."""
    name, n, L, seed = "nfw_512x512_64", 512, 100.0, 3000 + int(seed_offset)
    rng = np.random.default_rng(seed)
    if n_override is not None:
        n = int(n_override)
        name += "_n%d" % n
    x_min, y_min, dx = grid(n, L)
    out = np.empty((64, 6))
    for k in range(2):
        out[k] = (rng.uniform(-20, 20), rng.uniform(-20, 20), rng.uniform(0.0, 0.2), rng.uniform(0.0, np.pi),
                  rng.uniform(0.15, 0.3), rng.uniform(40.0, 80.0))
    for k in range(2, 64):
        while True:
            xc, yc = rng.normal(0.0, 40.0, 2)
            if abs(xc) < L and abs(yc) < L:
                break
        out[k] = (xc, yc, rng.uniform(0.0, 0.2), rng.uniform(0.0, np.pi), rng.uniform(0.02, 0.08), rng.uniform(1.0, 5.0))
    return Workload(name, out, x_min, y_min, dx, n, n, seed)
