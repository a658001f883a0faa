"""Generates the polynomial coefficients pasted into lt_math.cuh (atan(z)/z and atanh(z)/z on reduced ranges).

Near-minimax by interpolation at Chebyshev nodes in t = z^2 (mpmath, 50 digits), converted to the monomial basis;
prints C arrays and the measured max relative error of the fp64-rounded (resp. fp32-rounded) polynomial.
CUDA-path only: the CPU oracle uses libm/libquadmath log and atan2 and shares nothing with this.

    python paper_1902_03252_b200/csrc/gen_poly_coeffs.py
"""
import mpmath as mp

mp.mp.dps = 50


def g_atan(t):
    if t == 0:
        return mp.mpf(1)
    z = mp.sqrt(t)
    return mp.atan(z) / z


def g_atanh(t):
    if t == 0:
        return mp.mpf(1)
    z = mp.sqrt(t)
    return mp.atanh(z) / z


def cheb_fit(g, tmax, n):
    """degree-n polynomial in t on [0, tmax] interpolating g at the n+1 Chebyshev nodes; monomial coefficients."""
    nodes = [tmax * (1 + mp.cos(mp.pi * (2 * k + 1) / (2 * (n + 1)))) / 2 for k in range(n + 1)]
    A = mp.matrix(n + 1, n + 1)
    b = mp.matrix(n + 1, 1)
    for i, t in enumerate(nodes):
        for j in range(n + 1):
            A[i, j] = t ** j
        b[i] = g(t)
    c = mp.lu_solve(A, b)
    return [c[j] for j in range(n + 1)]


def max_err(g, tmax, coeffs, rnd):
    cs = [mp.mpf(rnd(c)) for c in coeffs]
    worst = mp.mpf(0)
    for k in range(2001):
        t = tmax * k / 2000
        p = mp.mpf(0)
        for c in reversed(cs):
            p = p * t + c
        worst = max(worst, abs(p / g(t) - 1))
    return worst


def f32(c):
    import numpy as np
    return float(np.float32(float(c)))


def emit(name, g, zmax, n, rnd, suffix):
    tmax = mp.mpf(zmax) ** 2
    c = cheb_fit(g, tmax, n)
    c[0] = mp.mpf(1)            # exact limit at 0 keeps the e -> 0 (circular) case exact
    err = max_err(g, tmax, c, rnd)
    print("// %s: degree %d in t=z^2, |z| <= %s, max rel err %s" % (name, n, mp.nstr(mp.mpf(zmax), 8), mp.nstr(err, 3)))
    print("static const %s %s[%d] = {%s};" % ("double" if suffix == "" else "float", name, n + 1,
                                               ", ".join(("%.17e" % rnd(x)) + suffix for x in c)))


if __name__ == "__main__":
    # table-driven range reductions of lt_math.cuh (eighth-octave bins chosen from the operands' bit patterns: half a
    # bin, 1/16 octave, plus the 0.0861 octave by which the piecewise-linear log2 of two bit patterns can be off) leave
    # |z| <= (r - 1)/(r + 1), r = 2^0.1486, i.e. 0.0515 for both atan and atanh; fitted on |z| <= 0.053
    zr = mp.mpf('0.053')
    for n in (3, 4, 5):
        emit("LT_ATAN_P64_%d" % n, g_atan, zr, n, float, "")
    for n in (3, 4, 5):
        emit("LT_ATANH_P64_%d" % n, g_atanh, zr, n, float, "")
    for n in (1, 2, 3):
        emit("LT_ATAN_P32_%d" % n, g_atan, zr, n, f32, "f")
    for n in (1, 2, 3):
        emit("LT_ATANH_P32_%d" % n, g_atanh, zr, n, f32, "f")
