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


def brute_drift(P, H, k0):
    K, M = P.shape
    S = np.zeros((K, M))
    for k in range(K):
        for r in range(M):
            for h in range(1, H + 1):
                kh, rh, t = k0 + h * (k - k0), h * r, h // 2
                if not (0 <= kh < K and rh < M):
                    continue
                S[k, r] += max(P[a, b] for a in range(max(0, kh - t), min(K, kh + t + 1))
                               for b in range(max(0, rh - t), min(M, rh + t + 1)))
    return S


def test_drift_tolerant_sum_brute_force_and_bounds():
    rng = np.random.default_rng(3)
    for K, M, k0 in ((7, 23, 3), (9, 40, 4), (1, 9, 0)):
        P = rng.standard_exponential((K, M))
        for H in (1, 2, 3, 5, 8):
            S = oh.harmonic_sum_drift(P, H, k0)
            np.testing.assert_allclose(S, brute_drift(P, H, k0), rtol=0, atol=1e-12)
            assert (S >= oh.harmonic_sum(P, H, k0) - 1e-12).all()           # a maximum over a window that holds the centre
    np.testing.assert_array_equal(oh.harmonic_sum_drift(P, 1, 0), P)


def test_drift_tolerant_sum_recovers_an_off_grid_pulse_train():
    # quantisation drifts the harmonics into adjacent bins.  Train at r0 = 3000.4, z = 4.6:
    # harmonic 3 sits at (13.8, 9001.2) -> cell (row of z = 14, bin 9001), not at 3 x (row of 4, 3000).
    w = workloads.harmonic_train(1 << 15, seed=1, r0=3000.4, z=4.6, power=50.0, rel_amplitudes=(1.0, 0.9, 0.8),
                                 zmax=20.0, dz=2.0, seglen=1024, noise=False)
    P = oracle.power_plane(w.spectrum, w.zmax, w.dz)
    k0 = oh.zero_row(w.zmax, w.dz)
    k1 = k0 + 2                                             # nearest row to z = 4.6 is z = 4
    peaks = [P[k0 + 2, 3000], P[k0 + 5, 6001], P[k0 + 7, 9001]]   # nearest cells of the three harmonics
    assert peaks[1] == P[k0 + 3:k0 + 6, 5999:6002].max() and peaks[2] == P[k0 + 5:k0 + 8, 8999:9002].max()
    Sd = oh.harmonic_sum_drift(P, 3, k0)
    Se = oh.harmonic_sum(P, 3, k0)
    assert abs(Sd[k1, 3000] - sum(peaks)) < 1e-9
    assert Se[k1, 3000] < 0.8 * Sd[k1, 3000]               # the exact-multiple sum misses the drifted harmonics
    assert np.unravel_index(np.argmax(Sd), Sd.shape) == (k1, 3000)
