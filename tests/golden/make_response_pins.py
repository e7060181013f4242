"""Writes tests/golden/response_centre_taps.txt.  Calls only oracle/ (never the CUDA path)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import numpy as np

import oracle

out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "response_centre_taps.txt")
with open(out, "w") as f:
    f.write("# written by tests/golden/make_response_pins.py from oracle/fdas_oracle.c\n")
    f.write("# (long-double Gauss-Legendre quadrature of W_z(q) = int_0^1 exp(2 pi i[q u + (z/2)(u^2-u)]) du)\n")
    f.write("# z  halfwidth  Re W_z(0)  Im W_z(0)  sum_j |h_z[j]|^2\n")
    for z in (2.0, 10.0, 20.0, 50.0, 96.0, 200.0):
        m = oracle.halfwidth(z)
        h = oracle.template_taps(z, m)
        w0 = np.conj(h[m])
        f.write(f"{z:g} {m} {w0.real:.15f} {w0.imag:.15f} {np.sum(np.abs(h) ** 2):.15f}\n")
print(open(out).read())
