"""GPU parity at the sizes bench.py times (BASELINE.json configs 3 and 4), in the launch configuration it times.

* config 3 (97 x 2^22 plane): EVERY bin of the fp32 planes (tensor-core split form and overlap-save FFT form)
  against the oracle's direct sum, every bin of the bf16 tensor-core plane against the oracle's direct sum over
  the bf16-rounded inputs, every bin of the bf16-stored plane against the oracle's rounding of that sum.  The
  oracle computes one plane row (2^22 bins) per call, so nothing here needs the fp64 plane in memory at once.
* config 4: one fdas_convolve_batched launch over a sub-batch of 32 series = 6.5e9 plane elements (26 GB): the
  32-bit row offsets, the 64-bit series base and the batch x K-row tensor map are exercised past 2^32 elements.
* the index kernels (fdas_peaks, fdas_harmonic_sum, fdas_harmonic_sum_drift, fdas_band_max) once on a seeded
  97 x 2^22 plane against their oracles (bit-exact / H 2^-23).

Tolerances are north_star's (fp32) and DESIGN.md section 7's (tensor-core accumulation), as in test_gpu_parity.
"""
import numpy as np
import pytest

import oracle
from oracle import bands as ob
from oracle import bf16 as obf
from oracle import harmonic as oh
from helpers import bf16_rne, z_values
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH, bf16_input_plane, check_fp32, check_mma   # noqa: F401  (F is a fixture)
from test_gpu_bf16_plane import bits_of, check_bf16_plane_bits

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def c3():
    return workloads.config3()


def _plane(F, w, precision, algorithm="auto", plane="f32"):
    import torch
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, precision, algorithm=algorithm, plane=plane)
    x = torch.from_numpy(np.ascontiguousarray(w.spectrum.astype(np.complex64))).cuda()
    P = plan.convolve(x)
    torch.cuda.synchronize()
    return plan, P


def test_config3_whole_plane_fp32_both_forms(F, c3):
    import torch
    w = c3
    planm, Pm = _plane(F, w, "f32")                       # AUTO = the split-operand tensor-core form bench.py times
    planf, Pf = _plane(F, w, "f32", algorithm="fft")
    assert planm.algorithm() == "mma" and planf.algorithm() == "fft" and tuple(Pm.shape) == (97, 1 << 22)
    p_peak = float(Pf.max().item())
    X = w.spectrum.astype(np.complex128)
    worst = {"mma": 0.0, "fft": 0.0}
    for k, z in enumerate(z_values(w.zmax, w.dz)):
        exp = oracle.convolve_row(X, oracle.template_taps(float(z)))          # all 2^22 bins of row k
        worst["mma"] = max(worst["mma"], check_fp32(Pm[k].cpu().numpy(), exp, p_peak)[0])
        worst["fft"] = max(worst["fft"], check_fp32(Pf[k].cpu().numpy(), exp, p_peak)[0])
    print(f"config3 whole plane: max |dP| split form {worst['mma']:.3e}, FFT form {worst['fft']:.3e} "
          f"(tolerance {1e-4 * p_peak + 1e-4:.3e})")
    del Pm, Pf
    torch.cuda.empty_cache()


def test_config3_whole_plane_bf16_tensor_core_form(F, c3):
    import torch
    w = c3
    plan, Pb = _plane(F, w, "bf16")
    plan16, P16 = _plane(F, w, "bf16", plane="bf16")
    assert plan.algorithm() == "mma" and plan16.algorithm() == "mma"
    p_peak = float(Pb.max().item())
    Xb = bf16_rne(w.spectrum.real).astype(np.float64) + 1j * bf16_rne(w.spectrum.imag).astype(np.float64)
    worst, off = 0.0, 0.0
    for k, z in enumerate(z_values(w.zmax, w.dz)):
        h = oracle.template_taps(float(z))
        hb = bf16_rne(h.real.astype(np.float32)).astype(np.float64) + 1j * bf16_rne(h.imag.astype(np.float32)).astype(np.float64)
        exp = oracle.convolve_row(Xb, hb)
        worst = max(worst, check_mma(Pb[k].cpu().numpy(), exp, p_peak)[0])
        off = max(off, check_bf16_plane_bits(bits_of(P16[k].contiguous()), exp, p_peak))
    print(f"config3 whole plane bf16: max |dP| {worst:.3e} (tolerance {1e-5 * p_peak + 1e-5:.3e}); "
          f"bf16-stored plane: at most {100 * off:.4f} % of a row off the oracle rounding (ties)")
    del Pb, P16
    torch.cuda.empty_cache()


@pytest.mark.parametrize("prec", ["bf16", "f32"])
def test_config4_sub_batch_of_32_crosses_2_to_32_elements(F, prec):
    import torch
    B = 32
    check = (0, 20, 31)                                   # series 20: element offset 20 x 97 x 2^21 = 4.07e9 > 2^32
    ws = {i: workloads.config4_series(i) for i in check}
    w0 = ws[0]
    X = np.empty((B, w0.M), dtype=np.complex64)
    for i in range(B):
        X[i] = ws[i].spectrum if i in ws else workloads.config4_series(i).spectrum
    plan = F.Plan(w0.N, w0.zmax, w0.dz, w0.seglen, prec)
    assert plan.algorithm() == "mma"
    Xd = torch.from_numpy(X).cuda()
    P = plan.convolve(Xd)
    torch.cuda.synchronize()
    assert tuple(P.shape) == (B, 97, 1 << 21) and P.numel() > (1 << 32)
    for i in check:
        single = plan.convolve(Xd[i].contiguous())
        assert torch.equal(single, P[i]), f"series {i}: batched and single-series planes differ"
        w = ws[i]
        s = int(w.injections[0].r0) - 2048 if w.injections else 777777
        p_peak = float(single.max().item())
        for s0 in (0, s, w.M - 4096):
            if prec == "bf16":
                check_mma(P[i, :, s0:s0 + 4096].cpu().numpy(), bf16_input_plane(w, s0, s0 + 4096), p_peak)
            else:
                check_fp32(P[i, :, s0:s0 + 4096].cpu().numpy(), oracle.power_plane(w.spectrum, w.zmax, w.dz, s0, s0 + 4096), p_peak)
        del single
    del P, Xd
    torch.cuda.empty_cache()


@pytest.fixture(scope="module")
def seeded_plane():
    """97 x 2^22 exponential noise with a few planted detections, plateaus and edge cells: an input
    of the index kernels that owes nothing to the CUDA path."""
    K, M = 97, 1 << 22
    rng = np.random.default_rng(33)
    P = rng.standard_exponential((K, M), dtype=np.float32)
    for k, r, v in [(0, 0, 40.0), (96, M - 1, 41.0), (48, 1 << 21, 60.0), (48, (1 << 21) + 1, 60.0), (49, 1 << 21, 60.0),
                    (10, 4095, 35.0), (10, 4096, 35.0), (96, 0, 33.0), (0, M - 1, 32.0), (47, 3000000, 55.0)]:
        P[k, r] = v
    # a pulse train on rows k0 + h (k - k0): harmonics 1..4 of (r = 250000, k = 52)
    for h in (1, 2, 3, 4):
        P[48 + 4 * h, 250000 * h] = 30.0 / h
    return P


def test_peaks_on_a_full_size_plane(F, seeded_plane):
    import torch
    P = seeded_plane
    plan = F.Plan(1 << 23, 96.0, 2.0, 2048, "f32")
    Pd = torch.from_numpy(P).cuda()
    thr = 17.0                                            # e^-17 x 4.07e8 ~ 17 noise cells + the planted ones
    n, rec = plan.peaks(Pd, thr)
    n_exp, rec_exp = oracle.peaks(P.astype(np.float64), thr)
    assert n == n_exp and n >= 10
    assert sorted((int(a), int(b), float(c)) for a, b, c in rec) == sorted(rec_exp)
    del Pd
    torch.cuda.empty_cache()


def test_harmonic_sum_and_band_max_on_a_full_size_plane(F, seeded_plane):
    import torch
    P = seeded_plane
    K, M = P.shape
    plan = F.Plan(1 << 23, 96.0, 2.0, 2048, "f32")
    Pd = torch.from_numpy(P).cuda()
    k0 = oh.zero_row(96.0, 2.0)
    P64 = P.astype(np.float64)
    H = 4                                                 # the harmonic count bench.py times
    S = plan.harmonic_sum(Pd, H).cpu().numpy()
    exp = oh.harmonic_sum(P64, H, k0)
    err = np.abs(S.astype(np.float64) - exp)
    assert (err <= H * 2.0 ** -23 * np.abs(exp) + 1e-30).all()
    assert abs(float(S[52, 250000]) - 30.0 * (1 + 1 / 2 + 1 / 3 + 1 / 4)) < 1e-4      # the planted train, gathered
    del exp
    # drift-tolerant form on a window of bins (its oracle is a python loop over the window cells): max is exact
    Sd = plan.harmonic_sum(Pd, H, drift=True).cpu().numpy()
    lo, n_r = 249000, 2048
    sub = oh.harmonic_sum_drift(P64[:, : H * (lo + n_r) + 8], H, k0)[:, lo:lo + n_r]
    errd = np.abs(Sd[:, lo:lo + n_r].astype(np.float64) - sub)
    assert (errd <= H * 2.0 ** -23 * np.abs(sub) + 1e-30).all()
    del P64, Sd, S
    # band maxima (Table 3): bit-exact, first maximum in (k, r) order
    for f_bin, nb in ((250000.0, 8), (1234.5, 32), (3.0e6, 4)):
        got = plan.band_max(Pd, f_bin, nb)
        assert got == ob.band_max(P, f_bin, nb)
    del Pd
    torch.cuda.empty_cache()
