"""Form Q: the dPIE deflection from the *definition* (alpha = grad psi, psi from kappa: eq. 2-4), as a 1-D
quadrature over the elliptically stratified surface density, in mpmath multi-precision.  TEST INFRASTRUCTURE.

It shares no formula with lt_oracle.cpp's Form C (no complex log, no closed form): only the convergence
  kappa(rho^2) = (b0/2) rcut/(rcut-rcore) [1/sqrt(rcore^2+rho^2) - 1/sqrt(rcut^2+rho^2)],
  rho^2 = x^2/(1+e)^2 + y^2/(1-e)^2   (lens frame, major axis along x; reading R1)
and the textbook reduction of eq. 3 for a density constant on similar ellipses xi^2 = x^2 + y^2/q^2,
q = (1-e)/(1+e):
  alpha_x = q x J0,  alpha_y = q y J1,
  J_n = int_0^1 kappa(xi(u)^2) [1-(1-q^2)u]^-(n+1/2) du,   xi(u)^2 = u (x^2 + y^2/(1-(1-q^2)u)).
(For q = 1 this is alpha(R) = (2/R) int_0^R kappa(r) r dr, the circular Gauss law.)

Used to (a) pin the C++ oracle on tiny inputs, (b) write tests/golden/dpie_golden.txt (tests/golden/make_golden.py).
Slow: tiny inputs only.
"""
import mpmath as mp


def kappa_dpie(rho2, rcore, rcut, b0):
    return (b0 / 2) * rcut / (rcut - rcore) * (1 / mp.sqrt(rcore ** 2 + rho2) - 1 / mp.sqrt(rcut ** 2 + rho2))


def dpie_lens_frame(x, y, e, rcore, rcut, b0):
    """(alpha_x, alpha_y) of one dPIE lens at lens-frame point (x, y) by quadrature."""
    x, y, e, rcore, rcut, b0 = [mp.mpf(v) for v in (x, y, e, rcore, rcut, b0)]
    q = (1 - e) / (1 + e)
    one_m_q2 = 1 - q * q

    def integrand(n):
        def f(u):
            den = 1 - one_m_q2 * u
            xi2 = u * (x * x + y * y / den)
            rho2 = xi2 / (1 + e) ** 2
            return kappa_dpie(rho2, rcore, rcut, b0) * den ** (-(n + mp.mpf(1) / 2))
        return f

    # break points concentrate near u = 0, where kappa varies on the scale (rcore/R)^2
    R2 = x * x + y * y / (q * q) + mp.mpf(10) ** -60
    u0 = min(mp.mpf(1) / 2, (rcore * (1 + e)) ** 2 / R2)
    pts = [mp.mpf(0)]
    for s in (mp.mpf(1) / 16, mp.mpf(1) / 4, 1, 4, 16, 64, 256, 1024, 4096):
        if u0 * s < 1:
            pts.append(u0 * s)
    pts.append(mp.mpf(1))
    J0 = mp.quad(integrand(0), pts)
    J1 = mp.quad(integrand(1), pts)
    return q * x * J0, q * y * J1


def gradient_point(lenses, t1, t2):
    """Algorithm 1 skeleton around the quadrature body; lenses = rows (xc, yc, e, Phi, rcore, rcut, b0)."""
    G1 = mp.mpf(0)
    G2 = mp.mpf(0)
    for (xc, yc, e, phi, rcore, rcut, b0) in lenses:
        d1 = mp.mpf(t1) - mp.mpf(xc)
        d2 = mp.mpf(t2) - mp.mpf(yc)
        c, s = mp.cos(mp.mpf(phi)), mp.sin(mp.mpf(phi))
        xp = d1 * c + d2 * s
        yp = d2 * c - d1 * s
        gx, gy = dpie_lens_frame(xp, yp, e, rcore, rcut, b0)
        G1 += gx * c - gy * s
        G2 += gy * c + gx * s
    return G1, G2
