"""Pins for oracle/harmonic.py (harmonic sum): CPU only."""
import numpy as np
import pytest

import oracle
from oracle import harmonic as oh
from paper_2206_12205_b200 import workloads


def brute(P, H, k0):
    K, M = P.shape
    S = np.zeros((K, M))
    for k in range(K):
        for r in range(M):
            for h in range(1, H + 1):
                kh, rh = k0 + h * (k - k0), h * r
                if 0 <= kh < K and rh < M:
                    S[k, r] += P[kh, rh]
    return S


def test_brute_force_tiny_planes():
    rng = np.random.default_rng(0)
    for K, M, k0 in ((7, 23, 3), (5, 16, 2), (9, 40, 4), (1, 9, 0)):
        P = rng.standard_exponential((K, M))
        for H in (1, 2, 3, 5, 8):
            np.testing.assert_allclose(oh.harmonic_sum(P, H, k0), brute(P, H, k0), rtol=0, atol=1e-12)


def test_special_cases():
    rng = np.random.default_rng(1)
    P = rng.standard_exponential((11, 200))
    np.testing.assert_array_equal(oh.harmonic_sum(P, 1, 5), P)                 # H = 1: the plane itself
    S4 = oh.harmonic_sum(P, 4, 5)
    np.testing.assert_allclose(S4[5, :50], P[5, 0:200:1][:50] + P[5, 0:100:2][:50] + P[5, 0:150:3][:50] + P[5, 0:200:4][:50])
    np.testing.assert_allclose(S4[:, 0], [sum(P[5 + h * (k - 5), 0] for h in range(1, 5) if 0 <= 5 + h * (k - 5) < 11) for k in range(11)])
    # a single spike at harmonic 3 of (k0 + 1, 20) reaches exactly that cell, for H >= 3 only
    Q = np.zeros((11, 200)); Q[5 + 3, 60] = 7.0
    assert oh.harmonic_sum(Q, 2, 5)[6, 20] == 0.0 and oh.harmonic_sum(Q, 3, 5)[6, 20] == 7.0
    assert oh.harmonic_sum(Q, 3, 5).sum() == 14.0                              # itself (h = 1) and that cell
    # linear in the plane; symmetric grid mirror: S(P flipped in k) = S(P) flipped in k
    np.testing.assert_allclose(oh.harmonic_sum(2 * P + Q, 3, 5), 2 * oh.harmonic_sum(P, 3, 5) + oh.harmonic_sum(Q, 3, 5))
    np.testing.assert_allclose(oh.harmonic_sum(P[::-1], 4, 5), S4[::-1])
    assert oh.zero_row(96.0, 2.0) == 48 and oh.zero_row(20.0, 2.0) == 10
    with pytest.raises(ValueError):
        oh.zero_row(5.0, 2.0)


def test_noise_free_pulse_train_closed_form():
    # harmonics at integer multiples of f and fdot.  Train on the grid: r0 = 3000, z = 4,
    # harmonics h = 1, 2, 3 with relative amplitudes 1, 0.8, 0.5 -> peaks at (h z, h r0) of coherent power
    # p a_h^2 (sum |h_{hz}|^2)^2 each (pin P9); the harmonic sum gathers them in ONE cell (k(z), r0).
    w = workloads.harmonic_train(1 << 15, seed=1, r0=3000.0, z=4.0, power=50.0, rel_amplitudes=(1.0, 0.8, 0.5),
                                 zmax=20.0, dz=2.0, seglen=1024, noise=False)
    P = oracle.power_plane(w.spectrum, w.zmax, w.dz)
    k0 = oh.zero_row(w.zmax, w.dz)
    S = oh.harmonic_sum(P, 3, k0)
    k, r = np.unravel_index(np.argmax(S), S.shape)
    assert (k, r) == (k0 + 2, 3000)
    want = 0.0
    for h, a in ((1, 1.0), (2, 0.8), (3, 0.5)):
        e = float((np.abs(oracle.template_taps(4.0 * h)) ** 2).sum())
        want += 50.0 * a * a * e * e
    assert abs(S[k, r] - want) / want < 2e-3          # cross terms between the harmonics' sidelobes are O(1e-3)
    assert abs(S[k, r] - (P[k0 + 2, 3000] + P[k0 + 4, 6000] + P[k0 + 6, 9000])) < 1e-9
    # and it beats the brightest single harmonic by the expected margin
    assert S[k, r] > 1.8 * P.max()
