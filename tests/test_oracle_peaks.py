"""Pins for the oracle's peak rule (P15) -- tiny hand-built planes."""
import numpy as np

import oracle
from oracle import reference as ref


def both(P, thr):
    n, rec = oracle.peaks(P, thr)
    py = ref.peaks(np.asarray(P, dtype=float), thr)
    assert n == len(rec) == len(py)
    assert sorted(rec) == sorted(py)
    return sorted((k, r) for k, r, _ in rec)


def test_single_spike_and_threshold():
    P = np.zeros((5, 7))
    P[2, 3] = 9.0
    assert both(P, 1.0) == [(2, 3)]
    assert both(P, 9.0) == []            # strictly above threshold
    assert both(P, 8.999) == [(2, 3)]


def test_edges_and_corners_have_fewer_neighbours():
    P = np.zeros((3, 4))
    P[0, 0] = 5
    P[2, 3] = 6
    P[0, 3] = 7
    assert both(P, 1.0) == [(0, 0), (0, 3), (2, 3)]


def test_plateau_yields_exactly_one_peak():
    P = np.zeros((4, 6))
    P[1, 2] = P[1, 3] = P[2, 2] = 4.0     # connected plateau
    assert both(P, 1.0) == [(1, 2)]       # the lexicographically first cell
    Q = np.zeros((3, 5))
    Q[1, 1] = Q[1, 2] = 3.0               # two adjacent equal values
    assert both(Q, 1.0) == [(1, 1)]


def test_neighbour_dominates():
    P = np.zeros((3, 5))
    P[1, 1] = 3.0
    P[2, 2] = 3.5                          # diagonal neighbour is higher
    assert both(P, 1.0) == [(2, 2)]
    P[0, 4] = 2.0                          # not adjacent to either
    assert both(P, 1.0) == [(0, 4), (2, 2)]


def test_capacity_follows_snprintf_convention():
    P = np.zeros((2, 9))
    P[0, 1] = P[0, 4] = P[1, 7] = 2.0
    n, rec = oracle.peaks(P, 1.0, capacity=2)
    assert n == 3 and len(rec) == 2


def test_random_plane_against_brute_force():
    rng = np.random.default_rng(4)
    P = rng.exponential(size=(9, 300))
    P[3, 100:103] = 5.0                    # a tie run
    got = both(P, 2.0)
    K, M = P.shape
    exp = []
    for k in range(K):
        for r in range(M):
            v = P[k, r]
            if v <= 2.0:
                continue
            ok = True
            for kk in range(max(0, k - 1), min(K, k + 2)):
                for rr in range(max(0, r - 1), min(M, r + 2)):
                    if (kk, rr) == (k, r):
                        continue
                    if (kk, rr) < (k, r):
                        ok &= v > P[kk, rr]
                    else:
                        ok &= v >= P[kk, rr]
            if ok:
                exp.append((k, r))
    assert got == exp
