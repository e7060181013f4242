"""GPU parity of fdas_band_max (Table 3) against oracle/bands.py: index work, bit-exact."""
import numpy as np
import pytest

import oracle
from oracle import bands as ob
from oracle import bf16 as obf
from oracle import harmonic as oh
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F   # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("zmax,M,prec,f_bin,n_bands", [
    (20.0, 4096, "f32", 100.0, 8), (20.0, 4099, "f32", 100.3, 32), (96.0, 50000, "f32", 1234.56, 12),
    (8.0, 1501, "f64", 37.77, 6), (20.0, 4096, "f32", 5000.0, 4), (0.0, 1101, "f32", 2.0, 32)])
def test_band_max_on_seeded_planes(F, zmax, M, prec, f_bin, n_bands):
    import torch
    plan = F.Plan(2 * M, zmax, 2.0, 1024 if zmax <= 20 else 2048, prec, build=False)
    rng = np.random.default_rng(M)
    P = rng.standard_exponential((plan.K, M)).astype(np.float64 if prec == "f64" else np.float32)
    P[:, ::7] = np.round(P[:, ::7], 1)                     # plenty of exact ties
    got = plan.band_max(torch.from_numpy(P).cuda(), f_bin, n_bands)
    exp = ob.band_max(P, f_bin, n_bands)
    assert [(k, r) for k, r, _ in got] == [(k, r) for k, r, _ in exp]
    assert [np.float32(v) for _, _, v in got] == [np.float32(v) for _, _, v in exp]


def test_band_max_of_a_bf16_plane_with_ties(F):
    import torch
    plan = F.Plan(2 * 8192, 20.0, 2.0, 1024, "bf16", plane="bf16")
    rng = np.random.default_rng(8)
    bits = obf.bf16_plane(rng.standard_exponential((plan.K, plan.M)).astype(np.float32))   # coarse grid: many equal maxima
    Pd = torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    got = plan.band_max(Pd, 333.3, 16)
    exp = ob.band_max(obf.quick_cast(bits), 333.3, 16)
    assert got == [(k, r, float(np.float32(v))) for k, r, v in exp]


def test_harmonics_of_a_convolved_pulse_train(F):
    # the paper's use: fundamental known a priori, the n-th harmonic = maximum of the n-th band
    import torch
    w = workloads.harmonic_train(1 << 18, seed=6, r0=9000.0, z=6.0, power=60.0, rel_amplitudes=(1.0, 0.9, 0.8, 0.7),
                                 zmax=40.0, dz=2.0, seglen=1024)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    P = plan.convolve(torch.from_numpy(w.spectrum).cuda())
    k0 = oh.zero_row(w.zmax, w.dz)
    got = plan.band_max(P, 9000.0, 4)
    assert [(k, r) for k, r, _ in got] == [(k0 + 3 * h, 9000 * h) for h in (1, 2, 3, 4)]
    exp = ob.band_max(oracle.power_plane(w.spectrum, w.zmax, w.dz), 9000.0, 4)
    assert [(k, r) for k, r, _ in exp] == [(k, r) for k, r, _ in got]
    for (_, _, a), (_, _, b) in zip(got, exp):
        assert abs(a - b) <= 1e-4 * exp[0][2] + 1e-4


def test_band_max_errors(F):
    import torch
    plan = F.Plan(2 * 4096, 4.0, 2.0, 1024, "f32", build=False)
    P = torch.zeros((plan.K, plan.M), dtype=torch.float32, device="cuda")
    out = torch.zeros(3 * 40, dtype=torch.int32, device="cuda")
    assert F.fdas_band_max(plan._h, P.data_ptr(), 0.0, 2, out.data_ptr()) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_band_max(plan._h, P.data_ptr(), 10.0, 0, out.data_ptr()) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_band_max(plan._h, P.data_ptr(), 10.0, 33, out.data_ptr()) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_band_max(plan._h, 0, 10.0, 2, out.data_ptr()) == F.FDAS_ERR_INVALID_ARG
    assert plan.band_max(P, 10.0, 2) == [(0, 0, 0.0), (0, 16, 0.0)]          # all-zero plane: first cell of each band
