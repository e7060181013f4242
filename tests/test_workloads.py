"""Seeded input generator: shapes, determinism, normalisation."""
import numpy as np

from paper_2206_12205_b200 import workloads


def test_config1_shape_and_determinism():
    a = workloads.config1()
    b = workloads.config1()
    assert a.N == 1 << 16 and a.M == 32768 and a.K == 21 and a.seglen == 1024
    assert a.spectrum.dtype == np.complex64 and a.spectrum.shape == (32768,)
    assert np.array_equal(a.spectrum, b.spectrum)
    # unit mean noise power (analytic scale 1/sqrt(N), sigma = 1)
    p = np.abs(a.spectrum[100:9000]) ** 2
    assert 0.95 < p.mean() < 1.05
    # the injected tone stands ~80x above the noise in the raw spectrum? no: z = 20 smears it;
    # the raw spectrum near r0 carries ~100/20 per bin
    assert (np.abs(a.spectrum[9990:10011]) ** 2).sum() > 60


def test_config2_draws():
    w = workloads.config2()
    assert w.M == 1 << 19 and w.K == 97 and w.seglen == 2048 and len(w.injections) == 8
    for t in w.injections:
        assert 1000 <= t.r0 <= 5e5 and -90 <= t.z <= 90 and 30 <= t.power <= 300


def test_config4_series_rule():
    w0 = workloads.config4_series(0)
    w1 = workloads.config4_series(1)
    assert w0.N == 1 << 22 and len(w0.injections) == 1 and len(w1.injections) == 0
    assert w0.seed == 100 and w1.seed == 101
