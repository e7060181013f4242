"""Test-side statement of what the fp32 variant's tensor-core form sums (include/fdas.h,
FDAS_ALGO_MMA on FDAS_F32), built from the oracle only: every fp32 operand is split into two
bfloat16 terms, x = x1 + x2 + (residual <= 2^-18 |x|), x1 = bf16(x), x2 = bf16(x - x1), and the
three leading products x1 h1 + x1 h2 + x2 h1 are summed (fp64 here, fp32 on the device)."""
import numpy as np

import oracle
from oracle import bf16 as obf
from helpers import z_values


def split2(v):
    """fp32 array -> (v1, v2) bf16-valued fp32 arrays with v1 = bf16(v), v2 = bf16(v - v1); v - v1 is exact in fp32."""
    v = np.asarray(v, dtype=np.float32)
    v1 = obf.round_to_bf16(v)
    v2 = obf.round_to_bf16(v - v1)
    return v1, v2


def split2c(z):
    z = np.asarray(z, dtype=np.complex64)
    r1, r2 = split2(z.real)
    i1, i2 = split2(z.imag)
    return (r1.astype(np.float64) + 1j * i1.astype(np.float64)), (r2.astype(np.float64) + 1j * i2.astype(np.float64))


def split_plane(w, r0=0, r1=None):
    """|x1*h1 + x1*h2 + x2*h1|^2 for every template, by the oracle's direct sum (fp64)."""
    x1, x2 = split2c(w.spectrum)
    rows = []
    for z in z_values(w.zmax, w.dz):
        h1, h2 = split2c(oracle.template_taps(float(z)).astype(np.complex64))   # taps stored in fp32 first (reading A11)
        _, y11 = oracle.convolve_row(x1, h1, r0, r1, want_y=True)
        _, y12 = oracle.convolve_row(x1, h2, r0, r1, want_y=True)
        _, y21 = oracle.convolve_row(x2, h1, r0, r1, want_y=True)
        y = y11 + y12 + y21
        rows.append(y.real ** 2 + y.imag ** 2)
    return np.stack(rows)
