"""The 'Real FFT' ahead of the convolution (Fig. 1, :85) -- TEST INFRASTRUCTURE, NOT PRODUCT
CODE (only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline leg may import this).

Definition (readings A8, A9): for N real samples x[j],

    X[k] = (1 / sqrt(N)) * sum_{j=0..N-1} x[j] exp(-2 pi i j k / N),     k = 0 .. N/2 - 1

(bins 0..N/2-1 of the real-input DFT, Nyquist dropped; with unit-variance noise the mean noise power
per bin is 1).  ``spectrum`` evaluates it in fp64 with ``numpy.fft.rfft`` as the library primitive for
the DFT; ``spectrum_direct`` is the same sum written out (small N only), and the tests pin both
against closed forms.  PAPER.md:97: "the 0th bin is the sum of all elements of the timeseries".
"""
from __future__ import annotations

import numpy as np


def spectrum(x) -> np.ndarray:
    x = np.asarray(x, dtype=np.float64)
    N = len(x)
    return np.fft.rfft(x)[: N // 2] / np.sqrt(N)


def spectrum_direct(x) -> np.ndarray:
    x = np.asarray(x, dtype=np.float64)
    N = len(x)
    j = np.arange(N)
    out = np.empty(N // 2, dtype=np.complex128)
    for k in range(N // 2):
        ph = (j * k) % N                                   # exact integer phase reduction
        out[k] = np.sum(x * np.exp(-2j * np.pi * ph / N))
    return out / np.sqrt(N)
