"""Generates the polynomial coefficients pasted into lt_math.cuh (atan(z)/z and atanh(z)/z on reduced ranges).

Near-minimax by interpolation at Chebyshev nodes in t = z^2 (mpmath, 50 digits), converted to the monomial basis;
prints C arrays and the measured max relative error of the fp64-rounded (resp. fp32-rounded) polynomial.
The fp64 arrays the kernels use are the `_HI` ones: the leading coefficient is rounded to a double whose low 32 bits are
zero (it is then an immediate of the first FMA of the Horner chain, which so reads one constant register instead of two:
lt_math.cuh) and the lower coefficients are refitted around it with the constant term exactly 1.
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


def hi_only(x):
    """nearest double whose low word is zero (21 significant bits): encodable as an FP64 immediate"""
    import struct
    b = struct.unpack('<Q', struct.pack('<d', float(x)))[0]
    lo = b & 0xffffffff
    b = (b & ~0xffffffff) + (0x100000000 if lo >= 0x80000000 else 0)
    return struct.unpack('<d', struct.pack('<Q', b))[0]


def refit_below(g, tmax, n, top):
    """degree n with c0 = 1 and c_n = top fixed: (g - 1 - top t^n) / t interpolated at n - 1 Chebyshev nodes"""
    m = n - 1
    nodes = [tmax * (1 + mp.cos(mp.pi * (2 * k + 1) / (2 * m))) / 2 for k in range(m)]
    A = mp.matrix(m, m)
    b = mp.matrix(m, 1)
    for i, t in enumerate(nodes):
        for j in range(m):
            A[i, j] = t ** j
        b[i] = (g(t) - 1 - mp.mpf(top) * t ** n) / t
    c = mp.lu_solve(A, b)
    return [mp.mpf(1)] + [c[j] for j in range(m)] + [mp.mpf(top)]


def emit_hi(name, g, zmax, n):
    tmax = mp.mpf(zmax) ** 2
    top = hi_only(cheb_fit(g, tmax, n)[n])
    c = refit_below(g, tmax, n, top)
    err = max_err(g, tmax, c, float)
    print("// %s: degree %d in t=z^2, |z| <= %s, leading coefficient %s (low word zero), max rel err %s"
          % (name, n, mp.nstr(mp.mpf(zmax), 8), float(top).hex(), mp.nstr(err, 3)))
    print("static const double %s[%d] = {%s};" % (name, n + 1, ", ".join("%.17e" % float(x) for x in c)))


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
    emit_hi("LT_ATAN_P64_4_HI", g_atan, zr, 4)
    emit_hi("LT_ATANH_P64_4_HI", g_atanh, zr, 4)
    for n in (1, 2, 3):
        emit("LT_ATAN_P32_%d" % n, g_atan, zr, n, f32, "f")
    for n in (1, 2, 3):
        emit("LT_ATANH_P32_%d" % n, g_atanh, zr, n, f32, "f")
