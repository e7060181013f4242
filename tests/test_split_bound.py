"""CPU-only: the split-operand sum the fp32 tensor-core form evaluates stays far inside the fp32
tolerance of BASELINE.json (|dP| <= 1e-4 P_peak + 1e-4) -- oracle against oracle, no GPU."""
import numpy as np

import oracle
from paper_2206_12205_b200 import workloads
from split_terms import split2, split_plane


def test_two_term_split_is_exact_to_2_pow_minus_17():
    rng = np.random.default_rng(2)
    v = (rng.standard_normal(100000) * np.exp(rng.uniform(-20, 20, 100000))).astype(np.float32)
    v1, v2 = split2(v)
    resid = np.abs(v.astype(np.float64) - v1.astype(np.float64) - v2.astype(np.float64))
    assert (resid <= np.abs(v) * 2.0 ** -17).all()
    assert (np.abs(v2) <= np.abs(v) * 2.0 ** -8).all()


def test_split_sum_against_the_plain_definition_config1():
    w = workloads.config1()
    exp = oracle.power_plane(w.spectrum, w.zmax, w.dz)
    got = split_plane(w)
    err = np.abs(got - exp)
    p_peak = exp.max()
    # dropped terms x2 h2, x3 h, x h3 are each <= 2^-17 |x h| and add incoherently over <= 53 taps
    assert err.max() <= 1e-5 * p_peak + 1e-5, err.max()
    assert (err / exp)[exp > 1].max() < 1e-4
    k, r = np.unravel_index(np.argmax(got), got.shape)
    assert (k, r) == (20, 10000)
