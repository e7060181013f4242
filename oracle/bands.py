"""Harmonic-band maxima of the f-fdot plane -- TEST INFRASTRUCTURE, NOT PRODUCT CODE (only tests/,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline leg may import this).

PAPER.md:186-199 (section 4.3, Table 3): "it is possible to preemptively split the f-fdot output plane
with boundaries (Table 3) derived from the fundamental frequency f ... the n-th harmonic is taken to
be the highest point in the n-th band."  Table 3:

    Fundamental       [0, 1.5 f]
    First harmonic    [1.5 f, 2.5 f]
    N-th harmonic     [(N + 0.5) f, (N + 1.5) f]

"[a, b] represents the closed interval inclusive of the upper bound, and lower in the case of the
fundamental": band 0 holds the bins 0 <= r <= 1.5 f, band N >= 1 the bins (N + 0.5) f < r <= (N + 1.5) f.
Here f is given in Fourier bins (f_bin = f T).  A band reaches over every row (all z) of the plane.
Ties (the paper is silent): the first cell in (k, r) lexicographic order.  An empty band (beyond the
plane) yields (-1, -1, 0).
"""
from __future__ import annotations

import math

import numpy as np


def band_bounds(f_bin: float, band: int, M: int):
    """(r_first, r_last) of band `band`, clipped to the plane; r_first > r_last when empty."""
    lo = 0 if band == 0 else int(math.floor((band + 0.5) * f_bin)) + 1
    hi = min(int(math.floor((band + 1.5) * f_bin)), M - 1)
    return lo, hi


def band_max(P, f_bin: float, n_bands: int):
    P = np.asarray(P)
    K, M = P.shape
    out = []
    for n in range(n_bands):
        lo, hi = band_bounds(f_bin, n, M)
        if lo > hi:
            out.append((-1, -1, 0.0))
            continue
        sub = P[:, lo:hi + 1]
        k, c = np.unravel_index(int(np.argmax(sub)), sub.shape)      # first maximum in (k, r) order
        out.append((int(k), int(lo + c), float(sub[k, c])))
    return out
