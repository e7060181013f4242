"""GPU parity of fdas_spectrum (the fp32 real FFT of PAPER.md:85, Fig. 1) against oracle/spectrum.py.

Tolerance: an fp32 FFT of N points carries a relative rms error of about
eps sqrt(log2 N) with eps = 2^-24 and a worst bin a few times that; the bound asserted is
|dX[k]| <= 8 eps log2(N) rms|X| + 2 eps |X[0]| on every bin: rms over the bins k >= 1, plus the rounding
of the partial sums that carry a non-zero mean (the data "may not be centered on zero";
those partial sums share butterflies with the bins whose index has trailing zero bits).  The DC bin
itself is checked relative to its own size."""
import numpy as np
import pytest

from oracle import spectrum as osp
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH   # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def series(N, seed, tone=None, mean=0.0):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal(N).astype(np.float32) + np.float32(mean)
    if tone is not None:
        r0, a = tone
        x += (a * np.cos(2 * np.pi * r0 * np.arange(N) / N)).astype(np.float32)
    return x


def check(got, exp, N):
    rms = float(np.sqrt((np.abs(exp[1:]) ** 2).mean()))
    tol = 8 * 2.0 ** -24 * np.log2(N) * rms + 2 * 2.0 ** -24 * abs(exp[0])
    err = np.abs(got.astype(np.complex128) - exp)
    assert err[1:].max() <= tol, (err[1:].max(), tol)
    assert err[0] <= 8 * 2.0 ** -24 * np.log2(N) * max(abs(exp[0]), rms)
    return err[1:].max(), tol


@pytest.mark.parametrize("logn", [10, 11, 12, 13, 14, 15, 18, 20, 23])
def test_spectrum_matches_the_definition(F, logn):
    import torch
    N = 1 << logn
    x = series(N, seed=logn, tone=(N / 8 + 0.25, 0.05), mean=0.5 if logn % 2 else 0.0)
    plan = F.Plan(N, 4.0, 2.0, 256, "f32", build=False)
    X = plan.spectrum(torch.from_numpy(x).cuda()).cpu().numpy()
    err, tol = check(X, osp.spectrum(x), N)
    print(f"N=2^{logn}: max |dX| {err:.3e} (tol {tol:.3e})")


def test_spectrum_closed_forms_and_f64_widening(F):
    import torch
    N = 1 << 14
    plan = F.Plan(N, 4.0, 2.0, 256, "f32", build=False)
    imp = np.zeros(N, dtype=np.float32); imp[5] = 1.0
    X = plan.spectrum(torch.from_numpy(imp).cuda()).cpu().numpy()
    k = np.arange(N // 2)
    assert np.abs(X - np.exp(-2j * np.pi * 5 * k / N) / np.sqrt(N)).max() < 1e-8
    a, r = 0.25, 1000
    tone = (a * np.cos(2 * np.pi * r * np.arange(N) / N)).astype(np.float32)
    X = plan.spectrum(torch.from_numpy(tone).cuda()).cpu().numpy()
    assert abs(X[r] - a * np.sqrt(N) / 2) < 1e-5 * a * np.sqrt(N)
    X[r] = 0
    assert np.abs(X).max() < 1e-5 * a * np.sqrt(N)
    # FDAS_F64 plans receive the same fp32 result widened
    p64 = F.Plan(N, 4.0, 2.0, 256, "f64", build=False)
    x = series(N, 3)
    X32 = plan.spectrum(torch.from_numpy(x).cuda())
    X64 = p64.spectrum(torch.from_numpy(x).cuda())
    assert X64.dtype == torch.complex128 and torch.equal(X64.to(torch.complex64), X32)
    # sizes the four-step FFT does not take
    bad = F.Plan(2 * 5000, 4.0, 2.0, 256, "f32", build=False)
    t = torch.zeros(10000, dtype=torch.float32, device="cuda")
    o = torch.zeros(5000, dtype=torch.complex64, device="cuda")
    assert F.fdas_spectrum(bad._h, t.data_ptr(), o.data_ptr()) == F.FDAS_ERR_UNSUPPORTED
    assert F.fdas_spectrum(plan._h, 0, o.data_ptr()) == F.FDAS_ERR_INVALID_ARG


def test_time_series_to_peaks_through_the_library(F):
    # Fig. 1 end to end on the device: time series -> real FFT -> convolve + peaks; the injected tone is found
    import torch
    N = 1 << 16
    rng = np.random.default_rng(1)
    x = rng.standard_normal(N).astype(np.float32)
    inj = workloads.Injection(r0=10000.25, z=20.0, power=100.0, phi0=0.0)
    workloads._add_tone(x, inj.r0, inj.z, inj.power, inj.phi0)
    plan = F.Plan(N, 20.0, 2.0, 1024, "bf16")
    X = plan.spectrum(torch.from_numpy(x).cuda())
    P, n, rec = plan.search(X, THRESH)
    assert (20, 10000) in {(int(a), int(b)) for a, b, _ in rec}
    # same series through the harness FFT (what every other test feeds): planes agree to the bf16 rule
    P2 = plan.convolve(torch.from_numpy(workloads.spectrum_of(x)).cuda())
    assert float(((P - P2).abs() / P2).mean().item()) < 0.02


def test_search_from_the_time_series_on_the_host(F):
    # the paper's accelerated flow starts at the time series (Fig. 1, :85): host series in, peak list out, checked
    # against oracle.spectrum -> oracle.power_plane -> oracle.peaks on config 1
    import oracle
    w = workloads.config1(keep_series=True)
    X = osp.spectrum(w.series)
    exp = oracle.power_plane(X, w.zmax, w.dz)
    n_exp, rec_exp = oracle.peaks(exp, THRESH)
    for prec in ("f32", "bf16", "f64"):
        plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
        rec = np.zeros(256, dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
        n = plan.search_host_timeseries(w.series, THRESH, rec, 256)
        assert (20, 10000) in {(int(a), int(b)) for a, b, _ in rec[:n].tolist()}           # the injected tone
        if prec != "bf16":
            assert n == n_exp and sorted((int(a), int(b)) for a, b, _ in rec[:n].tolist()) == sorted((k, r) for k, r, _ in rec_exp)
            got = {(int(a), int(b)): float(c) for a, b, c in rec[:n].tolist()}
            for k, r, pw in rec_exp:
                assert abs(got[(k, r)] - pw) <= 1e-4 * exp.max() + 1e-4
        # the pipelined batched form returns the same list for every copy of the series
        B, cap = 3, 64
        xs = np.stack([w.series] * B)
        recs = np.zeros((B, cap), dtype=rec.dtype)
        counts = np.zeros(B, dtype=np.int32)
        plan.search_host_batched(xs, THRESH, recs, counts, cap, timeseries=True)
        for b in range(B):
            assert counts[b] == n and sorted(map(tuple, recs[b, :n].tolist())) == sorted(map(tuple, rec[:n].tolist()))
