"""Pins for the oracle's template (response) functions -- CPU only.

Pins P1-P6, P12 of DESIGN.md section 3.  The C oracle evaluates the defining
integral by long-double quadrature; oracle/reference.py uses the Fresnel closed form;
scipy.integrate.quad is a third, independent route.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate
from scipy.special import fresnel

import oracle
from oracle import reference as ref
from helpers import bf16_rne, eq2_percent, wrapped_bank_row, z_values

GOLD = os.path.join(os.path.dirname(__file__), "golden")
Z_SET = [0.0, 2.0, -2.0, 20.0, -20.0, 7.5, 50.0, 96.0, -96.0, 200.0]


def test_halfwidth_rule():
    # BASELINE.json configs: "half-width ceil(|z|/2)+16"; m_max = 26 / 64 / 116 for zmax 20 / 96 / 200
    assert oracle.halfwidth(20) == 26 and oracle.halfwidth(-96) == 64 and oracle.halfwidth(200) == 116
    assert oracle.halfwidth(0) == 16 and oracle.halfwidth(7.5) == 20 and oracle.halfwidth(-3) == 18
    for z in Z_SET:
        assert oracle.halfwidth(z) == ref.halfwidth(z)


@pytest.mark.parametrize("z", Z_SET)
def test_P1_quadrature_equals_fresnel_closed_form(z):
    a = oracle.template_taps(z)
    b = ref.template_taps(z)
    assert a.shape == b.shape == (2 * oracle.halfwidth(z) + 1,)
    assert np.abs(a - b).max() < 1e-12


def test_P1_fractional_q_and_third_route():
    for z, q in [(20.0, 0.25), (20.0, -7.75), (-20.0, 3.5), (96.0, 40.1), (7.5, -2.2), (200.0, 115.5)]:
        w = oracle.response(z, q)
        c = complex(ref.response_closed_form(z, q))
        assert abs(w - c) < 1e-12
        f = lambda u, part: getattr(np.exp(2j * np.pi * (q * u + 0.5 * z * (u * u - u))), part)
        re = integrate.quad(f, 0, 1, args=("real",), limit=2000, epsabs=1e-13, epsrel=1e-13)[0]
        im = integrate.quad(f, 0, 1, args=("imag",), limit=2000, epsabs=1e-13, epsrel=1e-13)[0]
        assert abs(w - complex(re, im)) < 1e-10


def test_P2_zero_drift_is_fourier_interpolation_kernel():
    # z = 0: W_0(q) = exp(i pi q) sinc(q): delta at integer q, textbook interpolation kernel otherwise
    h = oracle.template_taps(0.0)
    m = oracle.halfwidth(0.0)
    d = np.zeros(2 * m + 1, dtype=complex)
    d[m] = 1.0
    assert np.abs(h - d).max() < 1e-15
    for q in (0.25, -0.5, 3.3, -11.9):
        expect = np.exp(1j * np.pi * q) * math.sin(math.pi * q) / (math.pi * q)
        assert abs(oracle.response(0.0, q) - expect) < 1e-15


@pytest.mark.parametrize("z", [2.0, 20.0, 7.5, 96.0, 200.0])
def test_P3_symmetries(z):
    hp = oracle.template_taps(z)
    hm = oracle.template_taps(-z)
    assert np.abs(hp - hp[::-1]).max() < 1e-15          # h_z[-j] = h_z[j]
    assert np.abs(hm - np.conj(hp)).max() < 1e-15       # h_{-z} = conj(h_z)
    # hence equal captured energy for +z and -z (PAPER.md:287 sees a 6th-figure asymmetry
    # only because its templates are generated in fp32)
    assert abs(np.sum(np.abs(hp) ** 2) - np.sum(np.abs(hm) ** 2)) < 1e-15


def test_P3_P4_centre_taps_and_energies():
    rows = [l.split() for l in open(os.path.join(GOLD, "response_centre_taps.txt")) if not l.startswith("#")]
    assert len(rows) == 6
    for zs, ms, re, im, en in rows:
        z, m = float(zs), int(ms)
        assert m == oracle.halfwidth(z)
        # closed form at q = 0: Y = -sqrt(z/2), Z = +sqrt(z/2), C and S odd
        S_, C_ = fresnel(math.sqrt(z / 2.0))
        w0 = np.exp(-1j * np.pi * ((z / 4.0) % 2.0)) / math.sqrt(2 * z) * 2.0 * (C_ + 1j * S_)
        assert abs(w0 - complex(float(re), float(im))) < 1e-12
        h = ref.template_taps(z)
        assert abs(np.conj(h[m]) - w0) < 1e-12
        assert abs(np.sum(np.abs(h) ** 2) - float(en)) < 1e-12
        assert 0.998 < float(en) <= 1.0          # reading A6: no renormalisation, energy 0.998..1


def test_P5_parseval_of_the_response():
    # sum_k |W_z(q-k)|^2 = 1: Fourier coefficients of a unit-modulus function on [0,1]
    for z, q in [(20.0, 0.0), (20.0, 0.37), (-50.0, 0.5)]:
        k = np.arange(-4000, 4001)
        w = ref.response_closed_form(z, q - k)
        s = np.sum(np.abs(w) ** 2)
        assert abs(s - 1.0) < 2e-4      # tail ~ 1/(pi^2 k) sum -> slowly to 1
        k2 = np.arange(-40000, 40001)
        s2 = np.sum(np.abs(ref.response_closed_form(z, q - k2)) ** 2)
        assert abs(s2 - 1.0) < abs(s - 1.0)


def test_P6_fft_of_template_is_the_time_domain_chirp():
    # H_z[f] * S -> exp(-i pi z (u^2 - u)), u = f/S, as the half-width grows (PAPER.md:109
    # Fig. 3 / :285 "flat convolution templates": near-unit magnitude)
    z, S = 20.0, 4096
    u = np.arange(S) / S
    chirp = np.exp(-1j * np.pi * z * (u * u - u))
    prev = None
    for m, bound in [(26, 0.03), (100, 0.004), (400, 0.0007), (1600, 0.0002)]:
        H = wrapped_bank_row(ref.template_taps(z, m), S) * S
        rms = math.sqrt(np.mean(np.abs(H - chirp) ** 2))
        assert rms < bound
        assert prev is None or rms < prev
        prev = rms
    H = wrapped_bank_row(oracle.template_taps(20.0), 1024) * 1024
    assert 0.9 < np.abs(H).min() and np.abs(H).max() < 1.1


def test_P12_bf16_conversion_statistics_match_paper_table1():
    # PAPER.md:133-138 Table 1 (fixture tests/golden/paper_table1_bf16_template_stats.txt):
    # Eq. 2 relative difference of bf16 vs fp32 template elements: |.| < 2^-8 = 0.390625 %,
    # mean ~ 0, sigma ~ 0.153 %.  Reproduced on this build's (synthetic) bank with RNE rounding.
    paper = {}
    for l in open(os.path.join(GOLD, "paper_table1_bf16_template_stats.txt")):
        if l.startswith("#"):
            continue
        name, mean, sd, mx, mn = l.split()
        paper[name] = tuple(map(float, (mean, sd, mx, mn)))
    S = 2048
    bank = np.stack([wrapped_bank_row(ref.template_taps(float(z)), S) for z in z_values(96.0, 2.0)])
    for part, name in ((bank.real, "real"), (bank.imag, "imaginary")):
        s = part.astype(np.float32)
        s = s[s != 0]
        d = eq2_percent(bf16_rne(s), s)
        assert np.abs(d).max() < 0.390625 * 1.002      # RNE bound (truncation would reach 0.78)
        assert abs(d.mean()) < 0.01
        assert 0.14 < d.std() < 0.18
        p_mean, p_sd, p_max, p_min = paper[name]
        assert abs(d.std() - p_sd) < 0.02 and p_max < 0.390625 and p_min > -0.390625
        assert abs(d.max() - p_max) < 0.01 and abs(d.min() - p_min) < 0.01
