"""ctypes loader for the NFW oracle (oracle/lt_oracle_nfw.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/ and
__graft_entry__.smoke() may import this module.  A catalogue is a float64 array [n, 6]: (xc, yc, epsilon, Phi, kappa_s, rs)."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lt_oracle_nfw.cpp")
_LIB = os.path.join(_HERE, "liblt_oracle_nfw.so")

LONG_DOUBLE, DOUBLE, QUAD = 0, 1, 3


def build(force=False):
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp%d" % os.getpid()
    subprocess.run(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-o", tmp, _SRC, "-lquadmath", "-lm"],
                   check=True)
    os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        vp, ci, cd, cll = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong
        L.lt_oracle_nfw_gradient_grid.argtypes = [vp, ci, cd, cd, cd, ci, ci, ci, vp, ci, ci]
        L.lt_oracle_nfw_gradient_points.argtypes = [vp, ci, vp, vp, cll, ci, vp, ci]
        L.lt_oracle_nfw_potential_points.argtypes = [vp, ci, vp, vp, cll, vp]
        L.lt_oracle_nfw_kappa.argtypes = [cd, cd, cd]
        L.lt_oracle_nfw_kappa.restype = cd
        _lib = L
    return _lib


def _lenses(lenses):
    a = np.ascontiguousarray(np.asarray(lenses, dtype=np.float64).reshape(-1, 6))
    return a, a.shape[0]


def _pts(px, py):
    px = np.ascontiguousarray(px, dtype=np.float64).ravel()
    py = np.ascontiguousarray(py, dtype=np.float64).ravel()
    assert px.shape == py.shape
    return px, py


def gradient_grid(lenses, x_min, y_min, dx, nx, ny, precision=LONG_DOUBLE, n_threads=0, row_stride=1):
    a, n = _lenses(lenses)
    out = np.full((ny, nx, 2), np.nan, dtype=np.float64)
    rc = lib().lt_oracle_nfw_gradient_grid(a.ctypes.data, n, float(x_min), float(y_min), float(dx), int(nx), int(ny),
                                           int(precision), out.ctypes.data, int(n_threads), int(row_stride))
    if rc != 0:
        raise ValueError("lt_oracle_nfw_gradient_grid: bad argument")
    return out


def gradient_points(lenses, px, py, precision=LONG_DOUBLE, n_threads=0):
    a, n = _lenses(lenses)
    px, py = _pts(px, py)
    out = np.empty((px.size, 2), dtype=np.float64)
    rc = lib().lt_oracle_nfw_gradient_points(a.ctypes.data, n, px.ctypes.data, py.ctypes.data, px.size, int(precision),
                                             out.ctypes.data, int(n_threads))
    if rc != 0:
        raise ValueError("lt_oracle_nfw_gradient_points: bad argument")
    return out


def potential_points(lenses, px, py):
    a, n = _lenses(lenses)
    px, py = _pts(px, py)
    out = np.empty(px.size, dtype=np.float64)
    lib().lt_oracle_nfw_potential_points(a.ctypes.data, n, px.ctypes.data, py.ctypes.data, px.size, out.ctypes.data)
    return out


def kappa(R, kappa_s, rs):
    return float(lib().lt_oracle_nfw_kappa(float(R), float(kappa_s), float(rs)))


def as_rule_catalogue(lenses):
    """[n,6] NFW catalogue -> the [n,7] layout oracle.lt_oracle.mixed_flags reads (x, y and the scale 4 kappa_s rs as b0)."""
    a, n = _lenses(lenses)
    out = np.zeros((n, 7))
    out[:, 0], out[:, 1], out[:, 6] = a[:, 0], a[:, 1], 4.0 * a[:, 4] * a[:, 5]
    out[:, 4], out[:, 5] = 1.0, 2.0
    return out
