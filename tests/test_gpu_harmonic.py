"""GPU parity of fdas_harmonic_sum against oracle/harmonic.py.

The sum runs over values already in device memory, so the comparison is exact up to the order of
<= H fp32 additions: |dS| <= H * 2^-23 * S (fp64 planes: 2^-52)."""
import numpy as np
import pytest

import oracle
from oracle import bf16 as obf
from oracle import harmonic as oh
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def check_sum(got, exp, H, eps):
    err = np.abs(got.astype(np.float64) - exp)
    assert (err <= H * eps * np.abs(exp) + 1e-30).all(), float((err / np.maximum(exp, 1e-30)).max())


@pytest.mark.parametrize("K_zmax,M,prec", [(20.0, 4096, "f32"), (20.0, 4099, "f32"), (96.0, 10000, "bf16"), (8.0, 1501, "f64"),
                                            (0.0, 1101, "f32")])
def test_harmonic_sum_on_seeded_planes(F, K_zmax, M, prec):
    import torch
    plan = F.Plan(2 * M, K_zmax, 2.0, 1024 if K_zmax <= 20 else 2048, prec, build=False)
    K = plan.K
    rng = np.random.default_rng(M)
    P = rng.standard_exponential((K, M))
    P = P.astype(np.float64 if prec == "f64" else np.float32)
    Pd = torch.from_numpy(P).cuda()
    k0 = oh.zero_row(K_zmax, 2.0)
    for H in (1, 2, 3, 4, 8, 16):
        S = plan.harmonic_sum(Pd, H).cpu().numpy()
        check_sum(S, oh.harmonic_sum(P.astype(np.float64), H, k0), H, 2.0 ** -52 if prec == "f64" else 2.0 ** -23)


def test_harmonic_sum_of_a_bf16_plane(F):
    import torch
    plan = F.Plan(2 * 8192, 20.0, 2.0, 1024, "bf16", plane="bf16")
    K, M = plan.K, plan.M
    rng = np.random.default_rng(4)
    bits = obf.bf16_plane(rng.standard_exponential((K, M)).astype(np.float32))
    Pd = torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    for H in (1, 4):
        S = plan.harmonic_sum(Pd, H).cpu().numpy()
        check_sum(S, oh.harmonic_sum(obf.quick_cast(bits).astype(np.float64), H, oh.zero_row(20.0, 2.0)), H, 2.0 ** -23)


def test_pulse_train_is_gathered_into_one_detection(F):
    # convolve a noisy 4-harmonic pulse train, sum 4 harmonics, find the peak
    import torch
    w = workloads.harmonic_train(1 << 18, seed=6, r0=9000.0, z=6.0, power=14.0, rel_amplitudes=(1.0, 0.9, 0.8, 0.7),
                                 zmax=40.0, dz=2.0, seglen=1024)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    x = torch.from_numpy(w.spectrum).cuda()
    P = plan.convolve(x)
    S = plan.harmonic_sum(P, 4)
    k0 = oh.zero_row(w.zmax, w.dz)
    exp = oh.harmonic_sum(oracle.power_plane(w.spectrum, w.zmax, w.dz), 4, k0)
    got = S.cpu().numpy().astype(np.float64)
    # the plane itself is within the fp32 tolerance of the oracle; the sum of 4 such values within 4x that
    assert np.abs(got - exp).max() <= 4 * (1e-4 * exp.max() + 1e-4)
    k, r = np.unravel_index(np.argmax(got), got.shape)
    assert (k, r) == (k0 + 3, 9000) == tuple(np.unravel_index(np.argmax(exp), exp.shape))
    # no single harmonic reaches the threshold a 4-fold sum of noise would need, the sum does (the point of summing)
    assert float(P.max().item()) < 25.0 < got[k, r]
    n, rec = plan.peaks(S, 30.0)
    assert (k, r) in {(int(a), int(b)) for a, b, _ in rec}


def test_harmonic_sum_errors(F):
    import torch
    plan = F.Plan(2 * 4096, 5.0, 2.0, 1024, "f32", build=False)              # grid -5..3: z = 0 is not a row
    P = torch.zeros((plan.K, plan.M), dtype=torch.float32, device="cuda")
    S = torch.zeros_like(P)
    assert F.fdas_harmonic_sum(plan._h, P.data_ptr(), S.data_ptr(), 2) == F.FDAS_ERR_UNSUPPORTED
    plan2 = F.Plan(2 * 4096, 4.0, 2.0, 1024, "f32", build=False)
    P = torch.zeros((plan2.K, plan2.M), dtype=torch.float32, device="cuda")
    S = torch.zeros_like(P)
    assert F.fdas_harmonic_sum(plan2._h, P.data_ptr(), S.data_ptr(), 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_harmonic_sum(plan2._h, P.data_ptr(), S.data_ptr(), 33) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_harmonic_sum(plan2._h, 0, S.data_ptr(), 2) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_harmonic_sum(plan2._h, P.data_ptr(), S.data_ptr(), 2) == 0


@pytest.mark.parametrize("K_zmax,M,prec", [(20.0, 4096, "f32"), (20.0, 4099, "f32"), (8.0, 1501, "f64"), (0.0, 1101, "f32")])
def test_drift_tolerant_sum_on_seeded_planes(F, K_zmax, M, prec):
    import torch
    plan = F.Plan(2 * M, K_zmax, 2.0, 1024, prec, build=False)
    rng = np.random.default_rng(M + 1)
    P = rng.standard_exponential((plan.K, M)).astype(np.float64 if prec == "f64" else np.float32)
    Pd = torch.from_numpy(P).cuda()
    k0 = oh.zero_row(K_zmax, 2.0)
    for H in (1, 2, 3, 5, 8):
        S = plan.harmonic_sum(Pd, H, drift=True).cpu().numpy()
        check_sum(S, oh.harmonic_sum_drift(P.astype(np.float64), H, k0), H, 2.0 ** -52 if prec == "f64" else 2.0 ** -23)


@pytest.mark.parametrize("M", [8192, 20000, 20004, 4101])
def test_drift_tolerant_sum_of_a_bf16_plane(F, M):
    # bf16-stored planes: rows that are 16-byte aligned (M % 8 == 0) take eight elements per load, the others one; several
    # 1024-bin tiles, spans that start at bin 0 and end at the plane's last bin, windows clipped at the first / last rows
    import torch
    plan = F.Plan(2 * M, 20.0, 2.0, 1024, "bf16", plane="bf16", build=False)
    K = plan.K
    rng = np.random.default_rng(M + 7)
    bits = obf.bf16_plane(rng.standard_exponential((K, M)).astype(np.float32))
    Pd = torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    wide = obf.quick_cast(bits).astype(np.float64)
    k0 = oh.zero_row(20.0, 2.0)
    for H in (2, 4, 5, 8):
        S = plan.harmonic_sum(Pd, H, drift=True).cpu().numpy()
        check_sum(S, oh.harmonic_sum_drift(wide, H, k0), H, 2.0 ** -23)


def test_drift_tolerant_sum_gathers_an_off_grid_pulse_train(F):
    # harmonics drift into adjacent bins; the exact-multiple sum misses them, the window sum does not
    import torch
    w = workloads.harmonic_train(1 << 18, seed=9, r0=9000.4, z=6.6, power=16.0, rel_amplitudes=(1.0, 0.9, 0.8, 0.7),
                                 zmax=40.0, dz=2.0, seglen=1024)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16")
    P = plan.convolve(torch.from_numpy(w.spectrum).cuda())
    Sd = plan.harmonic_sum(P, 4, drift=True)
    Se = plan.harmonic_sum(P, 4)
    assert bool((Sd >= Se).all())
    k0 = oh.zero_row(w.zmax, w.dz)
    cell = (k0 + 3, 9000)                                   # nearest cell of (z = 6.6, r0 = 9000.4)
    exp = oh.harmonic_sum_drift(P.cpu().numpy().astype(np.float64), 4, k0)
    assert abs(float(Sd[cell]) - exp[cell]) <= 4 * 2.0 ** -23 * exp[cell]
    assert float(Sd[cell]) > 1.25 * float(Se[cell])
    # the detection stands out of the summed noise where no single harmonic reaches the single-plane threshold
    assert float(P.max().item()) < THRESH < float(Sd[cell])
    assert float(Sd[cell]) >= 0.99 * float(Sd[:, 8000:10000].max().item())
