"""Plane-free search (second half): fdas_search and
fdas_search_batched with a NULL plane must return exactly the peak set -- cells AND powers, bit for bit -- of the
call that writes a plane, on every shape the fused search is tested on, and the oracle's peaks where the oracle's
plane decides them (config 1)."""
import numpy as np
import pytest

import oracle
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def as_set(rec):
    return sorted(map(tuple, rec.tolist()))


def both(plan, x, thr, capacity=1 << 20):
    _, n_ref, rec_ref = plan.search(x, thr, capacity=capacity)
    none, n, rec = plan.search(x, thr, capacity=capacity, plane_free=True)
    assert none is None
    assert n == n_ref, (n, n_ref)
    assert as_set(rec) == as_set(rec_ref)
    return n


@pytest.mark.parametrize("prec", ["bf16", "f32"])
def test_plane_free_search_equals_search_with_a_plane(F, prec):
    import torch
    w = workloads.config2()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
    x = torch.from_numpy(w.spectrum).cuda()
    for thr in (THRESH, 12.0, 6.0):
        n = both(plan, x, thr)
        assert n >= (8 if thr == THRESH else 20)
    for _ in range(3):                                  # the two tile counters alternate; the flags clean themselves
        both(plan, x, THRESH)
    # snprintf convention and capacity 0
    _, n_all, _ = plan.search(x, 6.0, capacity=1 << 20)
    _, n7, rec7 = plan.search(x, 6.0, capacity=7, plane_free=True)
    assert n7 == n_all and len(rec7) == 7
    _, n0, rec0 = plan.search(x, 6.0, capacity=0, plane_free=True)
    assert n0 == n_all and len(rec0) == 0


@pytest.mark.parametrize("prec", ["bf16", "f32"])
def test_plane_free_search_with_every_tile_listed(F, prec):
    # threshold inside the noise: every tile is listed with both neighbours, the recheck launch does all the work
    import torch
    w = workloads.noise_only(1 << 18, seed=9, zmax=96.0, dz=2.0, seglen=2048)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
    x = torch.from_numpy(w.spectrum).cuda()
    n = both(plan, x, 2.0, capacity=1 << 22)
    assert n > 100000


def test_plane_free_search_asymmetric_grid_groups_and_ragged_sizes(F):
    import torch
    for N, zmax, dz, S in ((2 * 50001, 5.0, 2.0, 1024),       # asymmetric grid, odd M (the plane path stores with scalar stores)
                           (2 * 70001, 200.0, 2.0, 4096),     # K = 201: two template groups -> one cluster per work item
                           (2 * 70000, 200.0, 2.0, 4096),
                           (2 * 1501, 8.0, 2.0, 256),         # a dozen tiles, the last one ragged
                           (2 * 300, 4.0, 2.0, 256)):         # fewer tiles than CTAs
        w = workloads.noise_only(N, seed=21, zmax=zmax, dz=dz, seglen=S)
        plan = F.Plan(w.N, zmax, dz, S, "bf16")
        x = torch.from_numpy(w.spectrum).cuda()
        for thr in (7.0, 3.0):
            n = both(plan, x, thr)
        assert n > 10


def test_plane_free_search_finds_the_oracle_peaks_of_config1(F):
    import torch
    w = workloads.config1()
    exp = oracle.power_plane(w.spectrum, w.zmax, w.dz)
    n_exp, rec_exp = oracle.peaks(exp, THRESH)
    for prec in ("bf16", "f32"):
        plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
        x = torch.from_numpy(w.spectrum).cuda()
        _, n, rec = plan.search(x, THRESH, plane_free=True)
        assert (20, 10000) in {(int(a), int(b)) for a, b, _ in rec}          # the injected tone (z = +20, r0 = 10000.25)
        if prec == "f32":
            assert n == n_exp
            got = {(int(a), int(b)): float(c) for a, b, c in rec}
            for k, r, pw in rec_exp:
                assert abs(got[(k, r)] - pw) <= 1e-4 * exp.max() + 1e-4


def test_plane_free_search_batched(F):
    import torch
    idx = [0, 10, 3, 20]
    ws = [workloads.config4_series(i) for i in idx]
    w0 = ws[0]
    plan = F.Plan(w0.N, w0.zmax, w0.dz, w0.seglen, "bf16")
    X = torch.from_numpy(np.stack([w.spectrum for w in ws])).cuda()
    for thr in (THRESH, 12.0):                          # e^-12 x 2.0e8 cells: about 1200 noise peaks per series
        counts, rec = plan.search_batched(X, thr, capacity=4096)
        for b in range(len(idx)):
            _, n_ref, rec_ref = plan.search(X[b].contiguous(), thr, capacity=4096)
            assert counts[b] == n_ref and n_ref <= 4096
            assert as_set(rec[b, :n_ref]) == as_set(rec_ref)
    # with planes: the same lists, and the planes of fdas_convolve_batched
    P = torch.empty((len(idx), plan.K, plan.M), dtype=torch.float32, device="cuda")
    counts2, rec2 = plan.search_batched(X, 12.0, capacity=4096, planes=P)
    assert np.array_equal(counts2, counts)
    for b in range(len(idx)):
        assert as_set(rec2[b, :counts[b]]) == as_set(rec[b, :counts[b]])
    assert torch.equal(P, plan.convolve(X))


def test_plane_free_search_unsupported_plans(F):
    import torch
    w = workloads.noise_only(2 * 5001, seed=5, zmax=20.0, dz=2.0, seglen=1024)
    x = torch.from_numpy(w.spectrum).cuda()
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    for prec, kw in (("f32", {}),                          # M % 4 != 0: the fp32 plan runs the FFT kernels
                     ("f64", {}),
                     ("bf16", {"algorithm": "fft"}),
                     ("bf16", {"plane": "bf16"})):         # the bf16-stored plane has its own (rounded) peak set
        plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec, **kw)
        xx = x.to(torch.complex128) if prec == "f64" else x
        assert F.fdas_search(plan._h, xx.data_ptr(), 0, 5.0, 0, 0, cnt.data_ptr()) == F.FDAS_ERR_UNSUPPORTED
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16")
    assert F.fdas_search(plan._h, x.data_ptr(), 0, 5.0, 0, 0, 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_search_batched(plan._h, x.data_ptr(), 0, 0, 5.0, 0, 0, cnt.data_ptr()) == F.FDAS_ERR_INVALID_ARG


def test_plane_free_search_config3(F):
    import torch
    w = workloads.config3()
    x = torch.from_numpy(w.spectrum).cuda()
    for prec in ("bf16", "f32"):
        plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
        n = both(plan, x, THRESH, capacity=1 << 16)
        assert n >= 64
    torch.cuda.empty_cache()


@pytest.mark.parametrize("prec,N", [("bf16", 1 << 21), ("f32", 1 << 21), ("bf16", (1 << 21) + 2 * 12345)])
def test_search_host_scans_the_spectrum_in_chunks(F, prec, N):
    # fdas_search_host on a spectrum of 8 MB and more: the copy is split into chunks and every chunk is scanned by
    # its own launch as soon as the next one has landed (the accelerated section starts with the
    # host -> device copy).  Same peaks, bit for bit, as the search of the whole spectrum on the device; the ragged
    # size ends with a partial block and a partial tile.
    import torch
    w = workloads.noise_only(N, seed=21, zmax=20.0, dz=2.0, seglen=1024)
    sp = w.spectrum.copy()
    rng = np.random.default_rng(5)
    M = len(sp)
    for r0 in (3, 1023, 1024, M // 8 - 1, M // 8, M // 2 + 77, M - 2):     # bright bins on and beside chunk / block boundaries
        sp[r0] += np.complex64(12.0 * np.exp(2j * np.pi * rng.random()))
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
    assert sp.nbytes >= 8 << 20
    _, n_ref, rec_ref = plan.search(torch.from_numpy(sp).cuda(), THRESH, capacity=1 << 16)
    assert n_ref >= 7
    rec = np.zeros(1 << 16, dtype=rec_ref.dtype)
    for _ in range(2):
        n = plan.search_host(sp, THRESH, rec, 1 << 16)
        assert n == n_ref
        assert as_set(rec[:n]) == as_set(rec_ref)
    # the count and the first 1024 records come back in one copy, the rest (if any) in a second one: a threshold with
    # thousands of peaks, the snprintf convention on a capacity below and above that split, capacity 0
    _, n_low, rec_low = plan.search(torch.from_numpy(sp).cuda(), 9.0, capacity=1 << 16)
    assert 1024 < n_low < (1 << 16)
    n = plan.search_host(sp, 9.0, rec, 1 << 16)
    assert n == n_low and as_set(rec[:n]) == as_set(rec_low)
    for cap in (0, 5, 1024, 1025, 3000):
        small = np.zeros(max(cap, 1), dtype=rec_ref.dtype)
        assert plan.search_host(sp, 9.0, small, cap) == n_low
        assert set(as_set(small[:min(cap, n_low)])) <= set(as_set(rec_low))
        assert len(set(as_set(small[:min(cap, n_low)]))) == min(cap, n_low)
