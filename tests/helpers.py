"""Test-only helpers (numpy): bf16 round-to-nearest-even emulation, Eq. 2 metric, z grid."""
import math

import numpy as np


def bf16_rne(x):
    """Round fp32 values to bfloat16 (round-to-nearest-even), returned as fp32.
    bf16 = top 16 bits of fp32 (Fig. 2)."""
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    u = a.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    r = ((u + 0x7FFF + lsb) >> 16) << 16
    return r.astype(np.uint32).view(np.float32).reshape(a.shape)


def eq2_percent(b, s):
    """PAPER.md:113 Eq. 2: % = (b - s) / ((b + s)/2) * 100."""
    b = np.asarray(b, dtype=np.float64)
    s = np.asarray(s, dtype=np.float64)
    return (b - s) / ((b + s) / 2.0) * 100.0


def z_values(zmax, dz):
    K = 2 * int(math.floor(zmax / dz + 1e-9)) + 1
    return -zmax + dz * np.arange(K)


def wrapped_bank_row(taps, S):
    """Test-side construction of H = FFT(wrapped taps)/S (used only to check identities the
    method relies on, e.g. overlap-save == direct sum; independent of the CUDA builder)."""
    m = (len(taps) - 1) // 2
    h = np.zeros(S, dtype=np.complex128)
    for j in range(-m, m + 1):
        h[j % S] = taps[j + m]
    return np.fft.fft(h) / S
