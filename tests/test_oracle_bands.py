"""Pins for oracle/bands.py (Table 3): CPU only."""
import os

import numpy as np

import oracle
from oracle import bands as ob
from oracle import harmonic as oh
from paper_2206_12205_b200 import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_bounds_follow_table3():
    rows = [l.split() for l in open(os.path.join(GOLD, "paper_table3_bands.txt")) if l.strip() and not l.startswith("#")]
    assert rows[0] == ["0", "0", "1.5"] and rows[1] == ["1", "1.5", "2.5"] and rows[2] == ["2", "2.5", "3.5"]
    f, M = 100.0, 10000
    for n in range(6):
        lo, hi = ob.band_bounds(f, n, M)
        lower, upper = (0.0 if n == 0 else (n + 0.5) * f), (n + 1.5) * f
        assert hi == int(upper) and (hi <= upper < hi + 1)                    # upper bound inclusive
        assert lo == (0 if n == 0 else int(lower) + 1)                        # lower bound exclusive, except the fundamental
    # consecutive bands tile the axis: no bin twice, none skipped
    for f in (100.0, 100.3, 37.77, 2.0):
        covered = []
        for n in range(8):
            lo, hi = ob.band_bounds(f, n, 10 ** 6)
            covered += list(range(lo, hi + 1))
        assert covered == list(range(0, covered[-1] + 1))
    assert ob.band_bounds(100.0, 0, 120) == (0, 119)                           # clipped at the plane edge
    lo, hi = ob.band_bounds(100.0, 3, 120)
    assert lo > hi                                                             # beyond the plane: empty


def test_band_max_brute_force_and_ties():
    rng = np.random.default_rng(0)
    P = rng.standard_exponential((5, 400))
    got = ob.band_max(P, 41.3, 8)
    for n, (k, r, v) in enumerate(got):
        lo, hi = ob.band_bounds(41.3, n, 400)
        best = (-1, -1, -1.0)
        for kk in range(5):
            for rr in range(lo, hi + 1):
                if P[kk, rr] > best[2]:
                    best = (kk, rr, P[kk, rr])
        assert (k, r, v) == best
    Q = np.zeros((3, 50)); Q[2, 7] = Q[1, 9] = Q[1, 4] = 5.0
    assert ob.band_max(Q, 10.0, 1) == [(1, 4, 5.0)]                             # first in (k, r) order
    assert ob.band_max(Q, 10.0, 7)[5:] == [(-1, -1, 0.0), (-1, -1, 0.0)]       # bands beyond the plane


def test_each_harmonic_of_a_pulse_train_is_its_band_maximum():
    # the n-th harmonic is the highest point of the n-th band
    w = workloads.harmonic_train(1 << 15, seed=1, r0=3000.0, z=4.0, power=50.0, rel_amplitudes=(1.0, 0.8, 0.5),
                                 zmax=20.0, dz=2.0, seglen=1024, noise=False)
    P = oracle.power_plane(w.spectrum, w.zmax, w.dz)
    k0 = oh.zero_row(w.zmax, w.dz)
    got = ob.band_max(P, 3000.0, 3)
    assert [(k, r) for k, r, _ in got] == [(k0 + 2, 3000), (k0 + 4, 6000), (k0 + 6, 9000)]
    assert got[0][2] > got[1][2] > got[2][2]
