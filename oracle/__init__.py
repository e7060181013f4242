"""FDAS oracle package -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

``oracle/fdas_oracle.c`` is the oracle proper (plain C, fp64, direct sums; templates by
long-double quadrature of the defining integral).  ``oracle/reference.py`` is its numpy
twin (Fresnel closed form + ``numpy.convolve``).  This module compiles the C file with gcc
and exposes it through ctypes.  Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s
cpu_baseline / ``--impl reference`` legs may import it; the product package never does.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdas_oracle.c")
_LIB = os.path.join(_HERE, "libfdas_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/fdas_oracle.c -> oracle/libfdas_oracle.so (gcc -O2 -fopenmp).

    No -ffast-math and no -march flags: the summation order written in the C file is the
    order executed.
    """
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        L.fdas_oracle_halfwidth.argtypes = [ctypes.c_double]
        L.fdas_oracle_halfwidth.restype = ctypes.c_int
        L.fdas_oracle_num_threads.argtypes = []
        L.fdas_oracle_num_threads.restype = ctypes.c_int
        L.fdas_oracle_response.argtypes = [ctypes.c_double, ctypes.c_double, dp, dp]
        L.fdas_oracle_response.restype = None
        L.fdas_oracle_template.argtypes = [ctypes.c_double, ctypes.c_int, dp]
        L.fdas_oracle_template.restype = ctypes.c_int
        L.fdas_oracle_row.argtypes = [dp, ctypes.c_int64, dp, ctypes.c_int, ctypes.c_int64,
                                      ctypes.c_int64, dp, dp]
        L.fdas_oracle_row.restype = ctypes.c_int
        L.fdas_oracle_plane.argtypes = [dp, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_int64, ctypes.c_int64, dp]
        L.fdas_oracle_plane.restype = ctypes.c_int
        L.fdas_oracle_halfwidth_jerk.argtypes = [ctypes.c_double, ctypes.c_double]
        L.fdas_oracle_halfwidth_jerk.restype = ctypes.c_int
        L.fdas_oracle_response_jerk.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, dp]
        L.fdas_oracle_response_jerk.restype = None
        L.fdas_oracle_template_jerk.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int, dp]
        L.fdas_oracle_template_jerk.restype = ctypes.c_int
        L.fdas_oracle_peaks.argtypes = [dp, ctypes.c_int, ctypes.c_int64, ctypes.c_double, dp,
                                        ctypes.c_int64]
        L.fdas_oracle_peaks.restype = ctypes.c_int64
        L.fdas_oracle_peaks3.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int64, ctypes.c_double, dp, ctypes.c_int64]
        L.fdas_oracle_peaks3.restype = ctypes.c_int64
        _lib = L
    return _lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def halfwidth(z: float) -> int:
    return int(lib().fdas_oracle_halfwidth(float(z)))


def num_threads() -> int:
    return int(lib().fdas_oracle_num_threads())


def response(z: float, q: float) -> complex:
    """W_z(q) by long-double Gauss-Legendre quadrature of the defining integral."""
    re = ctypes.c_double()
    im = ctypes.c_double()
    lib().fdas_oracle_response(float(z), float(q), ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def template_taps(z: float, m: int | None = None) -> np.ndarray:
    """h_z[j] = conj(W_z(j)), j = -m..m, complex128."""
    if m is None:
        m = halfwidth(z)
    out = np.empty(2 * (2 * m + 1), dtype=np.float64)
    rc = lib().fdas_oracle_template(float(z), int(m), _dptr(out))
    if rc:
        raise RuntimeError(f"fdas_oracle_template rc={rc}")
    return out.view(np.complex128)


def _as_c128(X) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(X, dtype=np.complex128))


def convolve_row(X, taps, r_begin: int = 0, r_end: int | None = None, want_y: bool = False):
    """Direct-sum row: returns P[r_begin:r_end] (and Y if want_y)."""
    X = _as_c128(X)
    M = len(X)
    if r_end is None:
        r_end = M
    taps = np.ascontiguousarray(np.asarray(taps, dtype=np.complex128))
    m = (len(taps) - 1) // 2
    p = np.empty(r_end - r_begin, dtype=np.float64)
    y = np.empty(2 * (r_end - r_begin), dtype=np.float64) if want_y else None
    rc = lib().fdas_oracle_row(_dptr(X.view(np.float64)), M, _dptr(taps.view(np.float64)), m,
                               int(r_begin), int(r_end), _dptr(p),
                               _dptr(y) if want_y else None)
    if rc:
        raise RuntimeError(f"fdas_oracle_row rc={rc}")
    return (p, y.view(np.complex128)) if want_y else p


def power_plane(X, zmax: float, dz: float, r_begin: int = 0, r_end: int | None = None) -> np.ndarray:
    """P[k][r - r_begin] for all K templates, float64 [K, r_end - r_begin]."""
    X = _as_c128(X)
    M = len(X)
    if r_end is None:
        r_end = M
    K = 2 * int(np.floor(zmax / dz + 1e-9)) + 1
    out = np.empty((K, r_end - r_begin), dtype=np.float64)
    rc = lib().fdas_oracle_plane(_dptr(X.view(np.float64)), M, float(zmax), float(dz),
                                 int(r_begin), int(r_end), _dptr(out))
    if rc:
        raise RuntimeError(f"fdas_oracle_plane rc={rc}")
    return out


def peaks(P, thr: float, capacity: int | None = None):
    """Returns (total_count, list of (k, r, power)) under the peak rule."""
    P = np.ascontiguousarray(np.asarray(P, dtype=np.float64))
    K, M = P.shape
    if capacity is None:
        capacity = int(np.count_nonzero(P > thr))
    out = np.empty(3 * max(capacity, 1), dtype=np.float64)
    n = int(lib().fdas_oracle_peaks(_dptr(P), K, M, float(thr), _dptr(out), int(capacity)))
    w = min(n, capacity)
    rec = [(int(out[3 * i]), int(out[3 * i + 1]), float(out[3 * i + 2])) for i in range(w)]
    return n, rec


# ---- jerk slab (reading A25) ---------------------------------------------
def halfwidth_jerk(z: float, w: float) -> int:
    return int(lib().fdas_oracle_halfwidth_jerk(float(z), float(w)))


def response_jerk(z: float, w: float, q: float) -> complex:
    re, im = ctypes.c_double(), ctypes.c_double()
    lib().fdas_oracle_response_jerk(float(z), float(w), float(q), ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def template_taps_jerk(z: float, w: float, m: int | None = None) -> np.ndarray:
    if m is None:
        m = halfwidth_jerk(z, w)
    out = np.empty(2 * (2 * m + 1), dtype=np.float64)
    rc = lib().fdas_oracle_template_jerk(float(z), float(w), int(m), _dptr(out))
    if rc:
        raise RuntimeError(f"fdas_oracle_template_jerk rc={rc}")
    return out.view(np.complex128)


def power_plane_jerk(X, zmax: float, dz: float, w: float, r_begin: int = 0, r_end: int | None = None) -> np.ndarray:
    """One slab of the f-fdot-fddot volume: the plane at jerk w, rows z_k = -zmax + k dz."""
    X = _as_c128(X)
    if r_end is None:
        r_end = len(X)
    K = 2 * int(np.floor(zmax / dz + 1e-9)) + 1
    return np.stack([convolve_row(X, template_taps_jerk(-zmax + k * dz, w), r_begin, r_end) for k in range(K)])


# ---- jerk volume (readings A25, A27) ----------------------------------------
def jerk_values(wmax: float, dw: float) -> np.ndarray:
    """w_i = -wmax + i dw, i = 0..2 floor(wmax/dw): the slabs of the volume (the same grid rule as z)."""
    n = int(np.floor(wmax / dw + 1e-9)) if dw > 0 else 0
    return -wmax + dw * np.arange(2 * n + 1)


def power_volume(X, zmax: float, dz: float, wmax: float, dw: float, r_begin: int = 0, r_end: int | None = None) -> np.ndarray:
    """V[i][k][r - r_begin]: the slab of every jerk value, float64 [W, K, r_end - r_begin]."""
    return np.stack([power_plane_jerk(X, zmax, dz, float(w), r_begin, r_end) for w in jerk_values(wmax, dw)])


def peaks3(V, thr: float, capacity: int | None = None):
    """Returns (total_count, list of (i, k, r, power)) under the 26-neighbour peak rule."""
    V = np.ascontiguousarray(np.asarray(V, dtype=np.float64))
    W, K, M = V.shape
    if capacity is None:
        capacity = int(np.count_nonzero(V > thr))
    out = np.empty(4 * max(capacity, 1), dtype=np.float64)
    n = int(lib().fdas_oracle_peaks3(_dptr(V), W, K, M, float(thr), _dptr(out), int(capacity)))
    w = min(n, capacity)
    rec = [(int(out[4 * i]), int(out[4 * i + 1]), int(out[4 * i + 2]), float(out[4 * i + 3])) for i in range(w)]
    return n, rec
