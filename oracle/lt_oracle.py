"""ctypes loader for the CPU oracle (oracle/lt_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_1902_03252_b200 and shares no code with the CUDA path.

Functions mirror the C entry points; see lt_oracle.cpp for the passages each follows (Algorithm 1 P:191-226,
eq. 24-28, BASELINE.json:north_star for the dPIE body).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lt_oracle.cpp")
_LIB = os.path.join(_HERE, "liblt_oracle.so")

LONG_DOUBLE, DOUBLE, FLOAT, QUAD = 0, 1, 2, 3

# DESIGN.md readings R11, R14, R15: (m_max, c28, patch half-width cluster ["], galaxy ["], b0 cluster threshold ["])
DEFAULT_MIXED = (3.26, 0.0104 / 0.03, 6.0, 0.3, 15.0)


def build(force=False):
    """Compile the oracle with g++ (-O2, no fast-math, OpenMP).  Building the checker is not using it."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-o", tmp, _SRC, "-lquadmath", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        L.lt_oracle_gradient_grid.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                              ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_void_p, ctypes.c_int, ctypes.c_int]
        L.lt_oracle_gradient_points.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                                ctypes.c_longlong, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                                ctypes.c_int]
        L.lt_oracle_kappa_points.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_longlong, ctypes.c_void_p]
        L.lt_oracle_mixed_flags.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                            ctypes.c_double, ctypes.c_double, ctypes.c_void_p, ctypes.c_int,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        L.lt_oracle_max_threads.restype = ctypes.c_int
        del dp
        _lib = L
    return _lib


def _lenses(lenses):
    a = np.ascontiguousarray(np.asarray(lenses, dtype=np.float64).reshape(-1, 7))
    return a, a.shape[0]


def max_threads():
    return int(lib().lt_oracle_max_threads())


def gradient_grid(lenses, x_min, y_min, dx, nx, ny, precision=LONG_DOUBLE, n_threads=0, row_stride=1):
    """Deflection map, shape [ny, nx, 2] fp64 (rows not on the stride stay NaN)."""
    a, n = _lenses(lenses)
    out = np.full((ny, nx, 2), np.nan, dtype=np.float64)
    rc = lib().lt_oracle_gradient_grid(a.ctypes.data, n, float(x_min), float(y_min), float(dx), int(nx), int(ny),
                                       int(precision), out.ctypes.data, int(n_threads), int(row_stride))
    if rc != 0:
        raise ValueError("lt_oracle_gradient_grid: bad argument")
    return out


def gradient_points(lenses, px, py, precision=LONG_DOUBLE, reflect=True, n_threads=0):
    """Deflection at arbitrary points; returns [npts, 2] fp64."""
    a, n = _lenses(lenses)
    px = np.ascontiguousarray(px, dtype=np.float64).ravel()
    py = np.ascontiguousarray(py, dtype=np.float64).ravel()
    assert px.shape == py.shape
    out = np.empty((px.size, 2), dtype=np.float64)
    rc = lib().lt_oracle_gradient_points(a.ctypes.data, n, px.ctypes.data, py.ctypes.data, px.size, int(precision),
                                         1 if reflect else 0, out.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError("lt_oracle_gradient_points: bad argument")
    return out


def kappa_points(lenses, px, py):
    a, n = _lenses(lenses)
    px = np.ascontiguousarray(px, dtype=np.float64).ravel()
    py = np.ascontiguousarray(py, dtype=np.float64).ravel()
    out = np.empty(px.size, dtype=np.float64)
    lib().lt_oracle_kappa_points(a.ctypes.data, n, px.ctypes.data, py.ctypes.data, px.size, out.ctypes.data)
    return out


def mixed_flags(sp_map, lenses, x_min, y_min, dx, mixed=DEFAULT_MIXED, want_crit=False):
    """Section 3.2-3.3 rule on a float32 map [ny, nx, 2].  Returns uint8 flags [ny, nx] (bit0 patch, bit1 eq.25,
    bit2 eq.28) and optionally the four criterion values [ny, nx, 4]."""
    sp = np.ascontiguousarray(sp_map, dtype=np.float32)
    ny, nx = sp.shape[0], sp.shape[1]
    a, n = _lenses(lenses)
    mp = np.asarray(mixed, dtype=np.float64)
    flags = np.zeros((ny, nx), dtype=np.uint8)
    crit = np.zeros((ny, nx, 4), dtype=np.float32) if want_crit else None
    rc = lib().lt_oracle_mixed_flags(sp.ctypes.data, nx, ny, float(x_min), float(y_min), float(dx), a.ctypes.data, n,
                                     mp.ctypes.data, flags.ctypes.data, crit.ctypes.data if want_crit else None)
    if rc != 0:
        raise ValueError("lt_oracle_mixed_flags: bad argument")
    return (flags, crit) if want_crit else flags


def mixed_map(lenses, x_min, y_min, dx, nx, ny, mixed=DEFAULT_MIXED, n_threads=0):
    """The paper's two-step mixed algorithm with the oracle on both steps: SP map = the reference map
    rounded to fp32 (an ideal SP pass), flags by the rule, flagged pixels take the reference fp64 value.
    Returns (map fp64 [ny,nx,2], flags)."""
    ref = gradient_grid(lenses, x_min, y_min, dx, nx, ny, LONG_DOUBLE, n_threads)
    sp = ref.astype(np.float32)
    flags = mixed_flags(sp, lenses, x_min, y_min, dx, mixed)
    out = sp.astype(np.float64)
    m = flags != 0
    out[m] = ref[m]
    return out, flags
