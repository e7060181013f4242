"""Pins for the jerk-volume oracle (readings A25, A27): the 26-neighbour peak rule on
hand-built volumes, against a sliced numpy twin and a pure-Python brute force, reduction to the plane rule, and an
injected (z, w) tone found in its own cell of the volume.  CPU only."""
import itertools

import numpy as np

import oracle
from oracle import reference as ref
from paper_2206_12205_b200 import workloads


def brute(V, thr):
    W, K, M = V.shape
    out = []
    for i, k, r in itertools.product(range(W), range(K), range(M)):
        v = V[i, k, r]
        if not v > thr:
            continue
        good = True
        for di, dk, dr in itertools.product((-1, 0, 1), repeat=3):
            if (di, dk, dr) == (0, 0, 0):
                continue
            a, b, c = i + di, k + dk, r + dr
            if not (0 <= a < W and 0 <= b < K and 0 <= c < M):
                continue
            n = V[a, b, c]
            if (a, b, c) < (i, k, r):          # precedes in (i, k, r) order: must be strictly smaller
                good &= bool(v > n)
            else:
                good &= bool(v >= n)
        if good:
            out.append((i, k, r, float(v)))
    return out


def all_three(V, thr):
    n, rec = oracle.peaks3(V, thr)
    tw = ref.peaks3(V, thr)
    assert n == len(rec) == len(tw)
    assert sorted(rec) == sorted(tw)
    return sorted((i, k, r) for i, k, r, _ in rec)


def test_hand_built_volumes():
    V = np.zeros((3, 4, 6))
    V[1, 2, 3] = 9.0
    assert all_three(V, 1.0) == [(1, 2, 3)]
    assert all_three(V, 9.0) == []                       # strictly above the threshold
    V[0, 1, 2] = 9.5                                     # a neighbour across the slab boundary (di = -1, dk = -1, dr = -1) dominates
    assert all_three(V, 1.0) == [(0, 1, 2)]
    V[2, 3, 5] = 4.0                                     # a corner of the volume: 7 neighbours only
    V[0, 0, 0] = 3.0
    assert all_three(V, 1.0) == [(0, 0, 0), (0, 1, 2), (2, 3, 5)]


def test_plateau_across_slabs_yields_one_peak():
    V = np.zeros((3, 3, 5))
    V[0, 1, 2] = V[1, 1, 2] = V[1, 2, 3] = 5.0           # connected through a slab step and a diagonal
    assert all_three(V, 1.0) == [(0, 1, 2)]              # the first cell in (i, k, r) order
    V = np.zeros((2, 2, 4))
    V[1, 0, 1] = V[0, 1, 2] = 2.0                        # equal values, adjacent across all three axes
    assert all_three(V, 1.0) == [(0, 1, 2)]


def test_single_slab_is_the_plane_rule():
    rng = np.random.default_rng(3)
    P = rng.exponential(size=(7, 200))
    P[3, 50:53] = 6.0
    n2, rec2 = oracle.peaks(P, 2.0)
    n3, rec3 = oracle.peaks3(P[None], 2.0)
    assert n2 == n3 and sorted(rec2) == sorted((k, r, v) for _, k, r, v in rec3)


def test_random_volume_against_brute_force():
    rng = np.random.default_rng(8)
    V = rng.exponential(size=(4, 6, 40))
    V[1, 2, 10:13] = 5.0                                  # tie runs along r, k and i
    V[2, 3:5, 20] = 5.5
    V[0:2, 5, 30] = 6.0
    n, rec = oracle.peaks3(V, 1.5)
    bf = brute(V, 1.5)
    assert n == len(bf) and sorted(rec) == sorted(bf) and sorted(ref.peaks3(V, 1.5)) == sorted(bf)
    n_all, few = oracle.peaks3(V, 1.5, capacity=3)       # snprintf convention
    assert n_all == n and len(few) == 3


def test_jerk_grid_and_volume_slabs():
    np.testing.assert_allclose(oracle.jerk_values(48.0, 24.0), [-48.0, -24.0, 0.0, 24.0, 48.0])
    np.testing.assert_allclose(oracle.jerk_values(0.0, 24.0), [0.0])
    np.testing.assert_allclose(oracle.jerk_values(30.0, 24.0), [-30.0, -6.0, 18.0])       # same rule as the z grid
    w = workloads.noise_only(1 << 12, seed=2, zmax=4.0, dz=2.0, seglen=256)
    V = oracle.power_volume(w.spectrum, 4.0, 2.0, 24.0, 24.0)
    assert V.shape == (3, 5, 2048)
    np.testing.assert_allclose(V[1], oracle.power_plane(w.spectrum, 4.0, 2.0), rtol=1e-12)     # the w = 0 slab is plain FDAS
    np.testing.assert_allclose(V[2], oracle.power_plane_jerk(w.spectrum, 4.0, 2.0, 24.0), rtol=0, atol=0)


def test_injected_jerk_tone_is_the_volume_peak_of_its_own_cell():
    # noise-free tone with z = 4, w = 36 on the (z, w) grid: the brightest cell of the volume is (w = 36, z = 4, r0)
    # with the closed-form power |A|^2 (sum |h_{z,w}|^2)^2 (pin P9 carried to the jerk response), and the volume
    # peak rule reports that cell -- in the w = 0 slab the same bin holds < 80 % of it
    wl = workloads.jerk_tone(1 << 15, seed=1, r0=4000.0, z=4.0, w=36.0, power=80.0, zmax=12.0, dz=2.0, seglen=1024, noise=False)
    V = oracle.power_volume(wl.spectrum, 12.0, 2.0, 36.0, 18.0, 3900, 4100)                # slabs w = -36, -18, 0, 18, 36
    i, k, r = np.unravel_index(np.argmax(V), V.shape)
    assert (i, k, r + 3900) == (4, 8, 4000)
    e = float((np.abs(oracle.template_taps_jerk(4.0, 36.0)) ** 2).sum())
    assert abs(V[i, k, r] - 80.0 * e * e) / (80.0 * e * e) < 2e-3
    n, rec = oracle.peaks3(V, 40.0)
    assert (4, 8, 100) in {(a, b, c) for a, b, c, _ in rec}
    assert V[2, 8, 100] < 0.8 * V[4, 8, 100]
    # symmetry of the volume: conjugating the spectrum's tone (z, w) -> (-z, -w) mirrors both axes
    wm = workloads.jerk_tone(1 << 15, seed=1, r0=4000.0, z=-4.0, w=-36.0, power=80.0, zmax=12.0, dz=2.0, seglen=1024, noise=False)
    Vm = oracle.power_volume(wm.spectrum, 12.0, 2.0, 36.0, 18.0, 3900, 4100)
    assert np.unravel_index(np.argmax(Vm), Vm.shape) == (0, 4, 100)
    assert abs(Vm.max() - V.max()) < 1e-6 * V.max()
