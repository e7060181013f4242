"""Pins for oracle/spectrum.py (the real FFT of PAPER.md Fig. 1, :85): CPU only."""
import numpy as np

from oracle import spectrum as osp
from paper_2206_12205_b200 import workloads


def test_direct_sum_equals_library_dft_small():
    rng = np.random.default_rng(0)
    for N in (8, 64, 250, 1024):
        x = rng.standard_normal(N)
        np.testing.assert_allclose(osp.spectrum(x), osp.spectrum_direct(x), rtol=0, atol=1e-12)


def test_closed_forms():
    N = 4096
    # bin 0 is the sum of all samples (scaled)
    x = np.random.default_rng(1).standard_normal(N) + 3.0
    assert abs(osp.spectrum(x)[0] - x.sum() / np.sqrt(N)) < 1e-10
    # impulse at j0: X[k] = exp(-2 pi i j0 k / N) / sqrt(N)
    imp = np.zeros(N); imp[5] = 1.0
    k = np.arange(N // 2)
    np.testing.assert_allclose(osp.spectrum(imp), np.exp(-2j * np.pi * 5 * k / N) / np.sqrt(N), atol=1e-14)
    # a cos(2 pi r j / N + phi) on bin r: X[r] = (a sqrt(N) / 2) e^{i phi}, every other bin 0  (|A|^2 = a^2 N / 4)
    a, r, phi = 0.3, 700, 0.4
    j = np.arange(N)
    X = osp.spectrum(a * np.cos(2 * np.pi * r * j / N + phi))
    assert abs(X[r] - a * np.sqrt(N) / 2 * np.exp(1j * phi)) < 1e-11
    X[r] = 0
    assert np.abs(X).max() < 1e-11
    # Parseval over the kept bins: sum_{k<N/2} |X|^2 = (sum x^2 + ...)/2 up to the DC and Nyquist terms
    x = np.random.default_rng(2).standard_normal(N)
    full = np.fft.fft(x) / np.sqrt(N)
    lhs = 2 * (np.abs(osp.spectrum(x)) ** 2).sum() - abs(full[0]) ** 2 + abs(full[N // 2]) ** 2
    assert abs(lhs - (x ** 2).sum()) < 1e-9
    # unit-variance noise: mean power per bin 1 (reading A9)
    big = np.random.default_rng(3).standard_normal(1 << 18)
    assert abs((np.abs(osp.spectrum(big)[1:]) ** 2).mean() - 1.0) < 0.01


def test_the_workload_generator_uses_this_definition():
    # workloads.spectrum_of is the fp32 harness FFT; it must agree with the fp64 definition to fp32 accuracy
    rng = np.random.default_rng(4)
    x = rng.standard_normal(1 << 14).astype(np.float32)
    d = np.abs(workloads.spectrum_of(x) - osp.spectrum(x)).max()
    assert d < 2e-5
