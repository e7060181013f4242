"""GPU parity of the f-fdot-fddot volume (fdas_volume_*, readings A25, A27): every slab
against oracle.power_volume with the plane tolerances, the 26-neighbour peak rule against oracle.peaks3 (index work:
same cells, same powers), and the injected (z, w) tone found by ONE library call."""
import numpy as np
import pytest

import oracle
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH, check_fp32, check_fp64   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def triples(rec):
    return sorted((int(a), int(b), int(c)) for a, b, c, _ in rec)


@pytest.fixture(scope="module")
def tone():
    return workloads.jerk_tone(1 << 16, seed=5, r0=9000.0, z=4.0, w=36.0, power=70.0, zmax=12.0, dz=2.0, seglen=1024)


@pytest.mark.parametrize("prec,algo", [("f64", "auto"), ("f32", "fft"), ("f32", "mma"), ("bf16", "mma"), ("bf16", "fft")])
def test_volume_slabs_match_the_oracle(F, tone, prec, algo):
    import torch
    w = tone
    vol = F.Volume(w.N, w.zmax, w.dz, 36.0, 18.0, w.seglen, prec, algorithm=algo)
    assert (vol.W, vol.K, vol.M) == (5, 13, 1 << 15)
    np.testing.assert_allclose(vol.w_values(), oracle.jerk_values(36.0, 18.0))
    x = torch.from_numpy(w.spectrum.astype(np.complex128 if prec == "f64" else np.complex64)).cuda()
    V = vol.convolve(x).cpu().numpy()
    exp = oracle.power_volume(w.spectrum, w.zmax, w.dz, 36.0, 18.0)
    if prec == "f64":
        check_fp64(V, exp)
    elif prec == "f32":
        check_fp32(V, exp)
    else:
        assert float((np.abs(V - exp) / exp).mean()) <= 0.02
        i, k, r = np.unravel_index(np.argmax(exp), exp.shape)
        assert abs(V[i, k, r] - exp[i, k, r]) <= 0.03 * exp[i, k, r]
    vol.close()


@pytest.mark.parametrize("prec", ["f64", "f32", "bf16"])
def test_volume_search_applies_the_26_neighbour_rule(F, tone, prec):
    import torch
    w = tone
    vol = F.Volume(w.N, w.zmax, w.dz, 36.0, 18.0, w.seglen, prec)
    x = torch.from_numpy(w.spectrum.astype(np.complex128 if prec == "f64" else np.complex64)).cuda()
    for thr in (THRESH, 9.0):
        V, n, rec = vol.search(x, thr)                      # ONE library entry: all slabs + volume peaks
        n_o, rec_o = oracle.peaks3(V.cpu().numpy().astype(np.float64), thr)
        assert n == n_o == len(rec)
        assert triples(rec.tolist()) == sorted((a, b, c) for a, b, c, _ in rec_o)
        got = {(int(a), int(b), int(c)): float(d) for a, b, c, d in rec.tolist()}
        for a, b, c, v in rec_o:
            assert got[(a, b, c)] == np.float32(v)
        n2, rec2 = vol.peaks(V, thr, capacity=3)            # snprintf convention
        assert n2 == n and len(rec2) == min(3, n)
    # the injected tone: slab w = 36 (index 4), z = 4 (row 8), r0 = 9000, and it is THE brightest record
    best = max(rec.tolist(), key=lambda t: t[3])
    assert tuple(int(t) for t in best[:3]) == (4, 8, 9000)
    if prec == "f64":
        # the oracle's own volume decides the same peaks (powers agree to 1e-10, no near-ties at this threshold)
        n_e, rec_e = oracle.peaks3(oracle.power_volume(w.spectrum, w.zmax, w.dz, 36.0, 18.0), THRESH)
        _, n, rec = vol.search(x, THRESH)
        assert n == n_e and triples(rec.tolist()) == sorted((a, b, c) for a, b, c, _ in rec_e)
    vol.close()


def test_volume_peak_rule_on_hand_built_volumes(F):
    import torch
    vol = F.Volume(2 * 1024, 4.0, 2.0, 24.0, 24.0, 256, "f32")     # W = 3, K = 5, M = 1024
    V = torch.zeros((3, 5, 1024), dtype=torch.float32, device="cuda")
    V[0, 1, 2] = V[1, 1, 2] = V[1, 2, 3] = 5.0                      # plateau through a slab step and a diagonal -> one peak
    V[0, 0, 0] = 4.0                                                # corners of the volume
    V[2, 4, 1023] = 6.0
    V[1, 3, 500] = 3.0
    V[2, 4, 501] = 3.5                                              # neighbour in the next slab dominates
    n, rec = vol.peaks(V, 1.0)
    assert triples(rec.tolist()) == [(0, 0, 0), (0, 1, 2), (2, 4, 501), (2, 4, 1023)]
    n_o, rec_o = oracle.peaks3(V.cpu().numpy(), 1.0)
    assert n == n_o and triples(rec.tolist()) == sorted((a, b, c) for a, b, c, _ in rec_o)
    assert vol.peaks(V, 6.0)[0] == 0                                # strictly above the threshold
    # odd M (scalar path of the kernel) and a single slab (the plane rule)
    vol1 = F.Volume(2 * 1001, 4.0, 2.0, 0.0, 24.0, 256, "f32")
    assert vol1.W == 1
    rng = np.random.default_rng(12)
    P = rng.standard_exponential((1, 5, 1001)).astype(np.float32)
    n, rec = vol1.peaks(torch.from_numpy(P).cuda(), 3.0)
    n_p, rec_p = oracle.peaks(P[0].astype(np.float64), 3.0)
    assert n == n_p and sorted((b, c) for _, b, c in triples(rec.tolist())) == sorted((k, r) for k, r, _ in rec_p)


def test_volume_host_entry_and_errors(F, tone):
    import torch
    w = tone
    vol = F.Volume(w.N, w.zmax, w.dz, 36.0, 18.0, w.seglen, "bf16")
    x = torch.from_numpy(w.spectrum).cuda()
    _, n_ref, rec_ref = vol.search(x, THRESH)
    rec = np.zeros(256, dtype=[("w_index", np.int32), ("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
    n = vol.search_host(w.spectrum, THRESH, rec, 256)
    assert n == n_ref and sorted(map(tuple, rec[:n].tolist())) == sorted(map(tuple, rec_ref.tolist()))
    assert vol.launch_count() > 5 * 4
    # errors: NULLs, bad grids, taps wider than the segment allows at |w| = wmax
    assert F.fdas_volume_convolve(vol._v, 0, 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_volume_w_of_index(vol._v, 5)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_volume_create(1 << 16, 12.0, 2.0, -1.0, 18.0, 1024, F.FDAS_F32)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_volume_create(1 << 16, 12.0, 2.0, 36.0, 0.0, 1024, F.FDAS_F32)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_volume_create(1 << 16, 96.0, 2.0, 1200.0, 600.0, 256, F.FDAS_F32)[0] == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_volume_destroy(None) == F.FDAS_OK
    vol.close()
