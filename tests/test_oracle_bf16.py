"""Pins for oracle/bf16.py (bf16 storage of the plane): CPU only."""
import os
from fractions import Fraction

import numpy as np
import pytest

from helpers import bf16_rne, eq2_percent
from oracle import bf16 as ob

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _table4():
    rows = []
    for l in open(os.path.join(GOLD, "paper_table4_powers.txt")):
        if l.startswith("#") or not l.strip():
            continue
        f = l.split()
        rows.append((f[0], float(f[1]), float(f[2]), float(f[3])))
    return rows


def test_paper_table4_bf16_powers_sit_on_the_bf16_grid():
    # the bfloat16 column is what a bf16-stored plane holds after the quick
    # cast, so every value must survive fp32 -> bf16 -> quick cast unchanged; the fp32 column
    # must not (it carries more than 8 significant bits), and the two agree within the paper's 3 %.
    for _, b, s, _ in _table4():
        assert ob.round_to_bf16(np.float32(b)) == np.float32(b)
        assert ob.round_to_bf16(np.float32(s)) != np.float32(s)
        assert abs(eq2_percent(b, s)) < 3.0


def test_quick_cast_is_byte_placement_and_exact():
    # PAPER.md:89 "appending 16x zero bits": value(bits) = value of the fp32 pattern bits << 16
    bits = np.array([0x0000, 0x8000, 0x3F80, 0xBF80, 0x4000, 0x3F81, 0x7F7F, 0x0001, 0x7F80, 0x4204], dtype=np.uint16)
    got = ob.quick_cast(bits)
    want = [0.0, -0.0, 1.0, -1.0, 2.0, 1.0 + 2.0 ** -7, (2 - 2.0 ** -7) * 2.0 ** 127, 2.0 ** -133, np.inf, 33.0]
    assert got.dtype == np.float32
    np.testing.assert_array_equal(got, np.array(want, dtype=np.float32))
    assert np.signbit(got[1])
    # low 16 bits of every result are zero
    assert not (got.view(np.uint32) & 0xFFFF).any()
    # all 65536 patterns: the fp32 pattern is bits << 16
    allb = np.arange(65536, dtype=np.uint32).astype(np.uint16)
    np.testing.assert_array_equal(ob.quick_cast(allb).view(np.uint32), allb.astype(np.uint32) << 16)


def test_rounding_special_cases_ties_to_even():
    f = np.float32
    cases = [
        (1.0, 0x3F80), (1.0 + 2.0 ** -8, 0x3F80),            # tie -> even (down)
        (1.0 + 3 * 2.0 ** -8, 0x3F82),                        # tie -> even (up)
        (1.0 + 2.0 ** -8 + 2.0 ** -23, 0x3F81),               # just above the tie
        (1.0 + 2.0 ** -8 - 2.0 ** -23 + 2.0 ** -7, 0x3F81),   # just below the next tie
        (-1.0 - 3 * 2.0 ** -8, 0xBF82),
        (2.0 - 2.0 ** -9, 0x4000),                            # carries into the exponent
        (0.0, 0x0000), (-0.0, 0x8000),
        (3.3895313892515355e38, 0x7F7F),                      # largest bf16
        (3.4028234663852886e38, 0x7F80),                      # fp32 max rounds to inf
        (np.inf, 0x7F80), (-np.inf, 0xFF80),
        (132.277, 0x4304), (48.777, 0x4243), (17.773, 0x418E),
    ]
    for x, want in cases:
        assert int(ob.to_bf16_bits(f(x))) == want, (x, hex(int(ob.to_bf16_bits(f(x)))), hex(want))
    assert np.isnan(ob.quick_cast(ob.to_bf16_bits(f(np.nan))))


def test_rounding_is_the_nearest_value_brute_force_with_exact_fractions():
    # independent of any float arithmetic: exact rational distance to both neighbours
    rng = np.random.default_rng(7)
    xs = np.concatenate([rng.standard_exponential(300).astype(np.float32) * 40,
                         rng.standard_normal(300).astype(np.float32),
                         (rng.standard_normal(100) * 1e-30).astype(np.float32),
                         np.array([1 + 2.0 ** -8, 1 + 3 * 2.0 ** -8, 257.0, 258.0, 259.0], dtype=np.float32)])
    got = ob.to_bf16_bits(xs)
    for x, g in zip(xs, got):
        lo = int(np.float32(x).view(np.uint32)) >> 16
        cands = [lo, lo + 1]
        vals = [Fraction(float(ob.quick_cast(np.uint16(c)))) for c in cands]
        d = [abs(Fraction(float(x)) - v) for v in vals]
        if d[0] < d[1]:
            want = cands[0]
        elif d[1] < d[0]:
            want = cands[1]
        else:
            want = cands[0] if cands[0] % 2 == 0 else cands[1]
        assert int(g) == want


def test_agrees_with_the_integer_trick_and_properties():
    rng = np.random.default_rng(11)
    x = np.concatenate([rng.standard_exponential(200000).astype(np.float32),
                        -rng.standard_exponential(1000).astype(np.float32) * 1e6,
                        np.linspace(0, 300, 100001, dtype=np.float32)])
    r = ob.round_to_bf16(x)
    np.testing.assert_array_equal(r, bf16_rne(x))                  # tests/helpers.py: add-and-shift form
    np.testing.assert_array_equal(ob.round_to_bf16(r), r)          # idempotent
    nz = x != 0
    rel = np.abs(r[nz].astype(np.float64) - x[nz]) / np.abs(x[nz].astype(np.float64))
    assert rel.max() <= 2.0 ** -8                                   # half an ulp of an 8-bit significand
    xs = np.sort(x)
    assert (np.diff(ob.round_to_bf16(xs)) >= 0).all()               # monotone
    # Table 1's bound: Eq. 2 difference within +-0.39 %
    assert np.abs(eq2_percent(r[nz], x[nz])).max() < 0.3922


def test_bf16_plane_of_exponential_noise_keeps_the_distribution():
    # "no change to the PDF" of the noise plane across precisions: mean and
    # variance of an exponential sample survive the rounding to well below sampling error.
    rng = np.random.default_rng(3)
    P = rng.standard_exponential(1 << 20).astype(np.float32)
    Q = ob.quick_cast(ob.bf16_plane(P))
    assert abs(Q.mean() / P.mean() - 1) < 2e-4
    assert abs(Q.var() / P.var() - 1) < 1e-3
