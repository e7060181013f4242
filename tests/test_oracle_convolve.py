"""Pins for the oracle's convolution / power plane -- CPU only (pins P2, P7, P9-P11)."""
import math

import numpy as np
import pytest

import oracle
from oracle import reference as ref
from helpers import wrapped_bank_row, z_values
from paper_2206_12205_b200 import workloads


def _rand_spectrum(M, seed):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal(M) + 1j * rng.standard_normal(M)) / math.sqrt(2.0)


def test_brute_force_tiny():
    # pure-Python double loop written from Y[r] = sum_j X[r-j] h[j], X = 0 outside [0, M)
    M = 37
    X = _rand_spectrum(M, 0)
    rng = np.random.default_rng(1)
    for m in (0, 1, 5, 18, 40):          # 40 > M: every tap range is clipped
        h = rng.standard_normal(2 * m + 1) + 1j * rng.standard_normal(2 * m + 1)
        Y = np.zeros(M, dtype=complex)
        for r in range(M):
            acc = 0j
            for j in range(-m, m + 1):
                if 0 <= r - j < M:
                    acc += X[r - j] * h[j + m]
            Y[r] = acc
        p, y = oracle.convolve_row(X, h, want_y=True)
        assert np.abs(y - Y).max() < 1e-13
        assert np.abs(p - np.abs(Y) ** 2).max() < 1e-12
        assert np.abs(ref.convolve_row(X, h) - Y).max() < 1e-13
        # windowed call returns the same numbers
        p2 = oracle.convolve_row(X, h, 5, 29)
        assert np.array_equal(p2, p[5:29])


def test_asymmetric_kernel_orientation():
    # a kernel that is NOT symmetric fixes convolution (X[r-j]) against correlation (X[r+j])
    X = np.zeros(16, dtype=complex)
    X[8] = 1.0
    h = np.array([1.0, 2.0, 3.0], dtype=complex)     # j = -1, 0, +1
    _, y = oracle.convolve_row(X, h, want_y=True)
    # Y[r] = h[r-8]: Y[7] = h[-1] = 1, Y[8] = 2, Y[9] = h[+1] = 3
    assert y[7] == 1 and y[8] == 2 and y[9] == 3


def test_P2_zero_drift_row_is_the_raw_power_spectrum():
    X = _rand_spectrum(500, 3)
    P = oracle.power_plane(X, 4.0, 2.0)               # z = -4,-2,0,2,4
    assert P.shape == (5, 500)
    assert np.abs(P[2] - (X.real ** 2 + X.imag ** 2)).max() < 1e-14


def test_c_oracle_equals_numpy_twin_plane():
    X = workloads.config1().spectrum[:4096]
    A = oracle.power_plane(X, 20.0, 2.0)
    B = ref.power_plane(X, 20.0, 2.0)
    assert A.shape == B.shape == (21, 4096)
    assert np.abs(A - B).max() < 1e-11 * max(1.0, A.max())
    W = oracle.power_plane(X, 20.0, 2.0, 1000, 1300)
    assert np.array_equal(W, A[:, 1000:1300])


@pytest.mark.parametrize("S,V,L", [(256, 200, 26), (256, 128, 64), (512, 460, 26), (1024, 960, 32)])
def test_P7_overlap_save_equals_direct_sum(S, V, L):
    # window the spectrum, circular-convolve each window by FFT, keep the
    # central region.  Window s covers X[sV-L .. sV-L+S-1]; outputs y[L+t], t < V, are valid
    # whenever L >= m and S - L - V >= m.  Any legal (S, V, L) gives the direct-sum result.
    M = 3000
    X = _rand_spectrum(M, 5)
    zmax = 20.0
    mmax = oracle.halfwidth(zmax)
    assert L >= mmax and S - L - V >= mmax
    P = oracle.power_plane(X, zmax, 2.0)
    nseg = -(-M // V)
    for k, z in enumerate(z_values(zmax, 2.0)):
        H = wrapped_bank_row(oracle.template_taps(float(z)), S)
        row = np.zeros(nseg * V)
        for s in range(nseg):
            idx = np.arange(s * V - L, s * V - L + S)
            seg = np.where((idx >= 0) & (idx < M), X[np.clip(idx, 0, M - 1)], 0)
            y = np.fft.ifft(np.fft.fft(seg) * H) * S      # unnormalised inverse; 1/S is in H
            row[s * V:(s + 1) * V] = np.abs(y[L:L + V]) ** 2
        assert np.abs(row[:M] - P[k]).max() < 1e-12 * max(1.0, P[k].max())


def test_P11_segment_parseval():
    S = 1024
    seg = _rand_spectrum(S, 9)
    F = np.fft.fft(seg)
    assert abs(np.sum(np.abs(F) ** 2) - S * np.sum(np.abs(seg) ** 2)) < 1e-9 * S * S
    H = wrapped_bank_row(oracle.template_taps(20.0), S)
    y = np.fft.ifft(F * H) * S
    assert abs(np.sum(np.abs(y) ** 2) - S * np.sum(np.abs(F) ** 2 * np.abs(H) ** 2)) < 1e-9 * S


def test_P9_config1_noise_free_worked_example():
    # Injected tone a = 2 sqrt(100/N), r0 = 10000.25, z = +20, no noise.  Peak in bin
    # (z = +20, r = 10000).  Ideal height 100 sinc^2(0.25) = 81.057 (scalloping);
    # exact truncated-template value |A sum_j W_z(r0 - r + j) h_z'[j]|^2.
    w = workloads.config1(noise=False)
    X = w.spectrum
    zs = z_values(20.0, 2.0)
    r_lo, r_hi = 9900, 10100
    P = oracle.power_plane(X, 20.0, 2.0, r_lo, r_hi)
    k, c = np.unravel_index(np.argmax(P), P.shape)
    assert zs[k] == 20.0 and r_lo + c == 10000
    peak = P[k, c]
    ideal = 100.0 * np.sinc(0.25) ** 2
    assert abs(peak - ideal) / ideal < 1e-3
    m = oracle.halfwidth(20.0)
    h = oracle.template_taps(20.0)
    pred = abs(10.0 * sum(oracle.response(20.0, 0.25 + j) * h[j + m] for j in range(-m, m + 1))) ** 2
    assert abs(peak - pred) / pred < 5e-5
    # sign of z (reading A3): the z = -20 row at the same bin holds only a few percent of it
    assert P[0, c] < 0.05 * peak
    # whole-plane closed form P[z'][r] ~ |A|^2 |W_{z-z'}(r0 - r)|^2 (infinite-template limit)
    for kk in (0, 5, 10, 15, 19, 20):
        for r in (9990, 9999, 10000, 10001, 10013):
            approx = 100.0 * abs(ref.response_closed_form(20.0 - zs[kk], 10000.25 - r)) ** 2
            assert abs(P[kk, r - r_lo] - approx) < 0.25 + 0.02 * approx


def test_P9_on_grid_tone_coherent_power():
    # integer r0, z on the grid: P_peak = |A|^2 (sum_j |h_z[j]|^2)^2
    N = 1 << 14
    x = np.zeros(N, dtype=np.float32)
    workloads._add_tone(x, 3000.0, -12.0, 64.0, 0.7)
    X = workloads.spectrum_of(x)
    P = oracle.power_plane(X, 20.0, 2.0, 2900, 3100)
    zs = z_values(20.0, 2.0)
    k, c = np.unravel_index(np.argmax(P), P.shape)
    assert zs[k] == -12.0 and 2900 + c == 3000
    e = np.sum(np.abs(oracle.template_taps(-12.0)) ** 2)
    assert abs(P[k, c] - 64.0 * e * e) / 64.0 < 2e-3     # negative-frequency image + fp32 series


def test_P10_noise_rows_are_exponential_with_mean_captured_energy():
    # Gaussian white input -> each row ~ exponential (chi^2_2 up to scale)
    from scipy import stats
    w = workloads.noise_only(1 << 17, seed=11, zmax=20.0)
    P = oracle.power_plane(w.spectrum, 20.0, 10.0)          # z = -20,-10,0,10,20
    n = P.shape[1]
    for k, z in enumerate(z_values(20.0, 10.0)):
        e = np.sum(np.abs(oracle.template_taps(float(z))) ** 2)
        row = P[k, 100:-100]
        assert abs(row.mean() - e) < 5.0 * e / math.sqrt(n / 4)
        # thin by the correlation length before the KS test
        d = stats.kstest(row[::64] / row.mean(), "expon")
        assert d.pvalue > 1e-3
