"""Harmonic sum over the f-fdot plane -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (only tests/,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline leg may import this).

What the paper fixes: "a pulsar with a given pulse frequency and acceleration
value will appear as a peak on this plane, with diminishing harmonics at integer multiples of both
f and fdot.  The summed height (power) of the peak and harmonics is typically used to calculate the
signal-to-noise ratio"; "a harmonic sum algorithm is used to gather the power from all harmonics
into a single detection".  The paper does not restate the algorithm of its reference (Adamek &
Armour 2018); the reading taken (A23) is the plain definition those two
sentences give:

    S_H[k][r] = sum_{h=1..H} P[k0 + h (k - k0)][h r],      k0 = row of z = 0,

a term being skipped when its row h (k - k0) + k0 falls outside 0..K-1 or its bin h r outside
0..M-1 (harmonic h of a signal at (r, z) sits at (h r, h z); z_k = (k - k0) dz, so h z_k is row
k0 + h (k - k0) exactly).  No drift tolerance: quantisation drift between harmonics
is left to the caller's peak rule.  Plain loops over h and k, numpy slicing over r.

``harmonic_sum_drift`` is the drift-tolerant form the paper motivates ("Quantisation
error in both the frequency and acceleration axes of the search lead to the observed peaks drifting
into adjacent bins.  To account for this, a harmonic sum algorithm is used").  Reading A26: a signal
found in cell (k, r) has true coordinates within half a cell, r_true = r + d, |d| <= 1/2 and likewise
in z, so its h-th harmonic lies within h/2 cells of (k0 + h (k - k0), h r); the sum takes, for every
h, the LARGEST power in that quantisation window:

    S'_H[k][r] = sum_{h=1..H}  max_{|dk| <= floor(h/2), |dr| <= floor(h/2)}  P[k0 + h (k - k0) + dk][h r + dr]

(cells outside the plane are skipped; a harmonic whose centre cell is outside the plane is skipped
altogether, as in the exact sum).  h = 1 has the window {0}: S'_1 = P.
"""
from __future__ import annotations

import numpy as np


def zero_row(zmax: float, dz: float) -> int:
    """Row k0 with z_k0 = 0 for the grid z_k = -zmax + k dz; raises if 0 is not on the grid."""
    n = int(np.floor(zmax / dz + 1e-9))
    if abs(n * dz - zmax) > 1e-9 * (1.0 + zmax):
        raise ValueError("z = 0 is not on the template grid: harmonics do not fall on rows")
    return n


def harmonic_sum(P, n_harmonics: int, k0: int) -> np.ndarray:
    P = np.asarray(P, dtype=np.float64)
    K, M = P.shape
    S = np.zeros_like(P)
    for h in range(1, int(n_harmonics) + 1):
        n_r = (M - 1) // h + 1                      # bins r with h r <= M - 1
        for k in range(K):
            kh = k0 + h * (k - k0)
            if 0 <= kh < K:
                S[k, :n_r] += P[kh, 0:h * (n_r - 1) + 1:h]
    return S


def harmonic_sum_drift(P, n_harmonics: int, k0: int) -> np.ndarray:
    P = np.asarray(P, dtype=np.float64)
    K, M = P.shape
    S = np.zeros_like(P)
    for h in range(1, int(n_harmonics) + 1):
        t = h // 2
        n_r = (M - 1) // h + 1
        for k in range(K):
            kh = k0 + h * (k - k0)
            if not 0 <= kh < K:
                continue
            best = np.full(n_r, -np.inf)
            for dk in range(-t, t + 1):
                if not 0 <= kh + dk < K:
                    continue
                for dr in range(-t, t + 1):
                    x = h * np.arange(n_r) + dr
                    ok = (x >= 0) & (x < M)
                    cand = np.full(n_r, -np.inf)
                    cand[ok] = P[kh + dk, x[ok]]
                    best = np.maximum(best, cand)
            S[k, :n_r] += best
    return S
