"""bfloat16 storage of the power plane and the paper's "quick cast" -- TEST INFRASTRUCTURE, NOT
PRODUCT CODE (only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline leg may
import this; it shares nothing with the CUDA library).

What the paper fixes (section 3.1, Fig. 2):

* a bfloat16 number is the sign, the 8 exponent bits and the top 7 fraction bits of an IEEE-754
  single: "in binary form a bfloat16 number can be represented in single-precision simply by
  appending 16x zero bits to the end";
* in the bfloat16 version of the pipeline the f-fdot plane is produced in bfloat16 and "the final
  cast to single-precision ... is completed by copying the two bytes of data for each bfloat16
  number into the corresponding positions of an all zero single-precision output array".

Rounding rule: round to nearest, ties to even (reading A12: Table 1's +-0.39 % = 2^-8
bound and ~0 mean, rule out truncation).

``to_bf16_bits`` is written as the *definition* -- of the two bf16 neighbours of x pick the nearer
one, on a tie the one whose last kept fraction bit is 0 -- in exact float64 arithmetic (every
fp32 and every bf16 value is exactly representable in float64), not as the usual integer
add-and-shift trick; ``tests/helpers.bf16_rne`` is that trick and the two pin each other.
"""
from __future__ import annotations

import numpy as np


def _bf16_floor_bits(x32: np.ndarray) -> np.ndarray:
    """Top 16 bits of the fp32 pattern = the bf16 neighbour of x towards zero."""
    return (np.ascontiguousarray(x32, dtype=np.float32).view(np.uint32) >> np.uint32(16)).astype(np.uint16)


def from_bf16_bits(bits) -> np.ndarray:
    """The "quick cast" of PAPER.md:91, literally: an all-zero single-precision array whose two
    most significant bytes receive the two bytes of each bfloat16 number (little endian host:
    bytes 2 and 3 of every 4-byte element)."""
    shape = np.shape(bits)
    b = np.ascontiguousarray(np.asarray(bits, dtype=np.uint16))
    out = np.zeros(b.shape, dtype=np.float32)
    ob = out.reshape(-1).view(np.uint8).reshape(-1, 4)
    ib = b.reshape(-1).view(np.uint8).reshape(-1, 2)
    ob[:, 2] = ib[:, 0]
    ob[:, 3] = ib[:, 1]
    return out.reshape(shape)


quick_cast = from_bf16_bits


def to_bf16_bits(x) -> np.ndarray:
    """fp32 -> bfloat16 bit patterns, round to nearest, ties to even (finite inputs and +-inf; NaN
    stays NaN).  Definition, not bit trick: candidates lo = x with the low 16 bits cleared (towards zero) and
    hi = the next bf16 value away from zero; the nearer wins; a tie goes to the candidate with an
    even 16-bit pattern."""
    shape = np.shape(x)
    x32 = np.ascontiguousarray(np.asarray(x, dtype=np.float32)).reshape(-1)
    lo_bits = _bf16_floor_bits(x32).astype(np.uint32)
    hi_bits = lo_bits + np.uint32(1)          # next magnitude: fraction + 1, carrying into the exponent (up to inf)
    lo = from_bf16_bits(lo_bits.astype(np.uint16)).astype(np.float64)
    with np.errstate(over="ignore", invalid="ignore"):
        hi = from_bf16_bits(hi_bits.astype(np.uint16)).astype(np.float64)
        x64 = x32.astype(np.float64)
        finite = np.isfinite(x64)
        # an overflowing candidate (inf) stands for 2^128 when measuring the distance (IEEE rule)
        hi_mag = np.where(np.isinf(hi), np.copysign(2.0 ** 128, hi), hi)
        d_lo = np.abs(x64 - lo)
        d_hi = np.abs(hi_mag - x64)
    take_hi = (d_hi < d_lo) | ((d_hi == d_lo) & ((lo_bits & 1) == 1))
    out = np.where(finite & take_hi, hi_bits, lo_bits).astype(np.uint16)
    nan = np.isnan(x64)
    if nan.any():
        out = np.where(nan, (lo_bits | np.uint32(0x40)).astype(np.uint16), out)   # keep it a (quiet) NaN
    return out.reshape(shape)


def round_to_bf16(x) -> np.ndarray:
    """fp32 -> nearest bf16 value, returned as fp32 (= quick_cast(to_bf16_bits(x)))."""
    return from_bf16_bits(to_bf16_bits(x))


def bf16_plane(P) -> np.ndarray:
    """The bf16-stored power plane of PAPER.md:91 as bit patterns: every power rounded once
    (RNE) from its fp32 value."""
    return to_bf16_bits(np.asarray(P, dtype=np.float32))
