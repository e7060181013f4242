"""numpy/scipy twin of the FDAS oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline leg may import
this.  It shares nothing with the CUDA library.

It states the same definition as ``oracle/fdas_oracle.c`` by a *different route*, so the
two can pin each other (tests/test_oracle_templates.py, pin P1):

* ``response_closed_form`` -- the constant-fdot Fourier response written with Fresnel
  integrals (the form Ransom et al. 2002 give; PAPER.md:37 cites it, PAPER.md:105 calls
  the result "a 1D array of complex numbers").  Derivation from the phase model of
  PAPER.md:53-57 (Eq. 1): complete the square in
  ``W_z(q) = int_0^1 exp(2 pi i [q u + (z/2)(u^2-u)]) du`` with ``q0 = q - z/2``,
  ``t = (u + q0/z) sqrt(2z)``:

      W_z(q) = exp(-i pi q0^2 / z) / sqrt(2z) * { [C(Z)-C(Y)] + i [S(Z)-S(Y)] },
      Y = q0 sqrt(2/z),  Z = (q0 + z) sqrt(2/z),      z > 0
      W_0(q) = exp(i pi q) sinc(q),      W_z(q) = conj(W_{-z}(-q)),  z < 0.

  (``scipy.special.fresnel`` is the library primitive for C and S.)
* ``template_taps`` -- h_z[j] = conj(W_z(j)), j = -m_z..m_z, m_z = ceil(|z|/2)+16
  (BASELINE.json configs).
* ``convolve_row`` -- Y_z[r] = sum_j X[r-j] h_z[j] via ``numpy.convolve`` (a direct sum),
  zero extension at the edges.
* ``power_plane`` / ``peaks`` -- P = |Y|^2 and the peak rule of DESIGN.md reading A14.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.special import fresnel


def halfwidth(z: float) -> int:
    """m_z = ceil(|z|/2) + 16 (BASELINE.json configs: "half-width ceil(|z|/2)+16")."""
    return int(math.ceil(abs(z) / 2.0)) + 16


def z_values(zmax: float, dz: float) -> np.ndarray:
    """z_k = -zmax + k dz, k = 0..K-1, K = 2 floor(zmax/dz) + 1 (SURVEY.md section 8 notation)."""
    K = 2 * int(math.floor(zmax / dz + 1e-9)) + 1
    return -zmax + dz * np.arange(K, dtype=np.float64)


def response_closed_form(z: float, q) -> np.ndarray:
    """W_z(q) for real q (array ok), Fresnel closed form (module docstring)."""
    q = np.asarray(q, dtype=np.float64)
    if z == 0.0:
        return np.exp(1j * np.pi * q) * np.sinc(q)
    if z < 0.0:
        return np.conj(response_closed_form(-z, -q))
    q0 = q - z / 2.0
    s = math.sqrt(2.0 / z)
    Y = q0 * s
    Z = (q0 + z) * s
    SZ, CZ = fresnel(Z)
    SY, CY = fresnel(Y)
    # phase exp(-i pi q0^2/z): reduce q0^2/z modulo 2 before multiplying by pi
    ph = np.mod(q0 * q0 / z, 2.0)
    return np.exp(-1j * np.pi * ph) / math.sqrt(2.0 * z) * ((CZ - CY) + 1j * (SZ - SY))


def template_taps(z: float, m: int | None = None) -> np.ndarray:
    """h_z[j] = conj(W_z(j)), j = -m..m (complex128, length 2m+1)."""
    if m is None:
        m = halfwidth(z)
    j = np.arange(-m, m + 1, dtype=np.float64)
    return np.conj(response_closed_form(z, j))


def convolve_row(X: np.ndarray, taps: np.ndarray) -> np.ndarray:
    """Y[r] = sum_{j=-m}^{m} X[r-j] h[j], r = 0..M-1, X zero outside [0, M)."""
    m = (len(taps) - 1) // 2
    full = np.convolve(np.asarray(X, dtype=np.complex128), taps)  # index n = r + m
    return full[m:m + len(X)]


def power_plane(X: np.ndarray, zmax: float, dz: float) -> np.ndarray:
    """P[k][r] = |Y_{z_k}[r]|^2, float64 [K, M]."""
    zs = z_values(zmax, dz)
    out = np.empty((len(zs), len(X)), dtype=np.float64)
    for k, z in enumerate(zs):
        y = convolve_row(X, template_taps(float(z)))
        out[k] = y.real ** 2 + y.imag ** 2
    return out


def peaks(P: np.ndarray, thr: float):
    """Peak rule (A14): P > thr, >= all 8 neighbours that exist, strictly > those
    that precede in (k, r) lexicographic order.  Returns a sorted list of (k, r, power)."""
    K, M = P.shape
    out = []
    for k in range(K):
        for r in np.nonzero(P[k] > thr)[0]:
            v = P[k, r]
            ok = True
            for dk in (-1, 0, 1):
                for dr in (-1, 0, 1):
                    if dk == 0 and dr == 0:
                        continue
                    kk, rr = k + dk, r + dr
                    if kk < 0 or kk >= K or rr < 0 or rr >= M:
                        continue
                    n = P[kk, rr]
                    precedes = dk < 0 or (dk == 0 and dr < 0)
                    if (not v > n) if precedes else (not v >= n):
                        ok = False
                        break
                if not ok:
                    break
            if ok:
                out.append((int(k), int(r), float(v)))
    return out


def peaks3(V: np.ndarray, thr: float):
    """Volume peak rule (A27) by another route than the C loops: a cell is a peak iff it exceeds thr and no
    existing cell of its 3 x 3 x 3 block beats it, where "beats" is > for cells after it in (i, k, r) order and >=
    for cells before it.  Written with array slices over the 26 offsets instead of per-cell loops."""
    V = np.asarray(V, dtype=np.float64)
    W, K, M = V.shape
    ok = V > thr
    pad = np.full((W + 2, K + 2, M + 2), -np.inf)
    pad[1:-1, 1:-1, 1:-1] = V
    for di in (-1, 0, 1):
        for dk in (-1, 0, 1):
            for dr in (-1, 0, 1):
                if di == dk == dr == 0:
                    continue
                nb = pad[1 + di:W + 1 + di, 1 + dk:K + 1 + dk, 1 + dr:M + 1 + dr]
                precedes = (di, dk, dr) < (0, 0, 0)
                ok &= (V > nb) if precedes else (V >= nb)
    return [(int(i), int(k), int(r), float(V[i, k, r])) for i, k, r in zip(*np.nonzero(ok))]
