"""Pins for the jerk-slab response of the oracle (reading A25): CPU only."""
import numpy as np
from scipy import integrate

import oracle
from paper_2206_12205_b200 import workloads


def quad_response(z, w, q):
    f = lambda u, part: getattr(np, part)(2 * np.pi * (q * u + 0.5 * z * (u * u - u) + (w / 12.0) * (2 * u ** 3 - 3 * u * u + u)))
    re = integrate.quad(f, 0, 1, args=("cos",), limit=2000, epsabs=1e-13, epsrel=1e-13)[0]
    im = integrate.quad(f, 0, 1, args=("sin",), limit=2000, epsabs=1e-13, epsrel=1e-13)[0]
    return complex(re, im)


def test_reduces_to_the_constant_acceleration_response():
    for z in (-20.0, 0.0, 7.5, 96.0):
        assert oracle.halfwidth_jerk(z, 0.0) == oracle.halfwidth(z)
        for q in (-3.0, 0.0, 0.25, 11.0):
            assert abs(oracle.response_jerk(z, 0.0, q) - oracle.response(z, q)) < 1e-15
        np.testing.assert_allclose(oracle.template_taps_jerk(z, 0.0), oracle.template_taps(z), atol=1e-15)


def test_against_adaptive_quadrature_and_symmetries():
    for z, w, q in ((4.0, 30.0, 2.0), (-10.0, 60.0, -5.0), (20.0, -45.0, 0.5), (0.0, 24.0, 1.0)):
        a = oracle.response_jerk(z, w, q)
        assert abs(a - quad_response(z, w, q)) < 1e-11
    for z, w in ((6.0, 40.0), (-12.0, 18.0)):
        for j in range(-9, 10):
            W = oracle.response_jerk(z, w, j)
            assert abs(oracle.response_jerk(z, -w, -j) - W) < 1e-14            # u -> 1 - u
            assert abs(oracle.response_jerk(-z, -w, -j) - np.conj(W)) < 1e-14   # complex conjugation
            assert abs(oracle.response_jerk(-z, w, j) - np.conj(W)) < 1e-14     # both: the +-z pairing survives a jerk
        h = oracle.template_taps_jerk(z, w)
        np.testing.assert_allclose(oracle.template_taps_jerk(-z, w), np.conj(h), atol=1e-14)
        assert np.abs(h - h[::-1]).max() > 1e-3                                  # but the taps are no longer even in j
    # width rule: largest excursion of the frequency from its mean is |z|/2 + |w|/12
    assert oracle.halfwidth_jerk(20.0, 60.0) == 10 + 5 + 16 and oracle.halfwidth_jerk(-3.0, -30.0) == 4 + 16
    # Parseval: sum_k |W(q - k)|^2 = 1; the truncated template keeps > 99 % of it
    for z, w in ((10.0, 48.0), (0.0, 96.0)):
        tot = sum(abs(oracle.response_jerk(z, w, k)) ** 2 for k in range(-400, 401))
        assert abs(tot - 1.0) < 2e-3
        assert (np.abs(oracle.template_taps_jerk(z, w)) ** 2).sum() > 0.99


def test_injected_jerk_signal_peaks_in_its_own_slab():
    # noise-free tone with z = 4, w = 36 on the grid: slab w = 36 holds |A|^2 (sum |h|^2)^2 at (z, r0);
    # the w = 0 slab (plain FDAS) misses part of the power
    w = workloads.jerk_tone(1 << 15, seed=1, r0=4000.0, z=4.0, w=36.0, power=80.0, zmax=12.0, dz=2.0, seglen=1024, noise=False)
    Pj = oracle.power_plane_jerk(w.spectrum, w.zmax, w.dz, 36.0, 3900, 4100)
    P0 = oracle.power_plane_jerk(w.spectrum, w.zmax, w.dz, 0.0, 3900, 4100)
    k, r = np.unravel_index(np.argmax(Pj), Pj.shape)
    assert (k, r + 3900) == (8, 4000)                                            # z = -12 + 2 k
    e = float((np.abs(oracle.template_taps_jerk(4.0, 36.0)) ** 2).sum())
    assert abs(Pj[k, r] - 80.0 * e * e) / (80.0 * e * e) < 2e-3
    assert P0.max() < 0.8 * Pj[k, r]
    np.testing.assert_allclose(P0, oracle.power_plane(w.spectrum, w.zmax, w.dz, 3900, 4100), rtol=1e-12)
