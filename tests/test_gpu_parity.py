"""GPU parity: libfdas (through the C ABI binding) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json north_star's:

  fp64 : relative error <= 1e-10 on every bin
  fp32 : |dP| <= 1e-4 * P_peak + 1e-4 on every bin
  bf16 : every above-threshold peak within 3 % of the fp32 peak power, in the same (z, r)
         bin or the adjacent z bin; mean relative power error <= 2 % over the plane
         (compared with the GPU fp32 plane, which is itself checked against the oracle)
"""
import math

import numpy as np
import pytest

import oracle
from helpers import bf16_rne, wrapped_bank_row, z_values
from paper_2206_12205_b200 import workloads

pytestmark = pytest.mark.gpu

THRESH = 22.5   # DESIGN.md reading A13: the paper's 44.982 in unit-mean-noise units


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_2206_12205_b200 import _build, fdas
    _build.build()
    fdas.lib()
    return fdas


def gpu_plane(F, w, precision, spectrum=None, algorithm="auto"):
    import torch
    X = w.spectrum if spectrum is None else spectrum
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, precision, algorithm=algorithm)
    dt = np.complex128 if precision == "f64" else np.complex64
    x = torch.from_numpy(np.ascontiguousarray(X.astype(dt))).cuda()
    P = plan.convolve(x)
    torch.cuda.synchronize()
    return plan, P


def check_fp64(got, exp):
    rel = np.abs(got - exp) / exp
    bad = int(np.count_nonzero(rel > 1e-10))
    assert bad == 0, f"{bad} bins above 1e-10, worst {rel.max():.3e} at P={exp.flat[np.argmax(rel)]:.3e}"


def check_fp32(got, exp, p_peak=None):
    if p_peak is None:
        p_peak = float(exp.max())
    tol = 1e-4 * p_peak + 1e-4
    err = np.abs(got.astype(np.float64) - exp)
    assert err.max() <= tol, f"max |dP| {err.max():.3e} > {tol:.3e}"
    return err.max(), tol


def bf16_input_plane(w, r0=0, r1=None):
    """What FDAS_ALGO_MMA computes, by the oracle: spectrum and taps rounded once to bf16 (RNE,
    DESIGN.md reading A12), then the plain fp64 direct sum (oracle.convolve_row)."""
    X = w.spectrum
    Xb = bf16_rne(X.real).astype(np.float64) + 1j * bf16_rne(X.imag).astype(np.float64)
    rows = []
    for z in z_values(w.zmax, w.dz):
        h = oracle.template_taps(float(z))
        hb = bf16_rne(h.real.astype(np.float32)).astype(np.float64) + \
            1j * bf16_rne(h.imag.astype(np.float32)).astype(np.float64)
        rows.append(oracle.convolve_row(Xb, hb, r0, r1))
    return np.stack(rows)


def check_mma(got, exp, p_peak=None):
    """fp32 accumulation of <= 2 (2 m_max + 1) <= 466 exact bf16 x bf16 products per component:
    |dY| <~ n eps |Y|-scale with eps = 2^-24, so |dP| <= 1e-5 P_peak + 1e-5 leaves > 10x margin
    (DESIGN.md section 7); a wrong tap, sign or index shows up at the 1e-2 .. 1 level."""
    if p_peak is None:
        p_peak = float(exp.max())
    tol = 1e-5 * p_peak + 1e-5
    err = np.abs(got.astype(np.float64) - exp)
    assert err.max() <= tol, f"max |dP| {err.max():.3e} > {tol:.3e}"
    return err.max(), tol


def check_bf16_rules(Pb, Pf, ref_peaks):
    """Pb, Pf: bf16 and fp32 planes (numpy, same shape); ref_peaks: (k, r, power) found in Pf."""
    K, M = Pf.shape
    rel = np.abs(Pb.astype(np.float64) - Pf) / Pf
    mean_rel = float(rel.mean())
    assert mean_rel <= 0.02, f"mean relative power error {mean_rel:.4f} > 2 %"
    worst = 0.0
    for k, r, pw in ref_peaks:
        # highest bf16 value in the same bin or the adjacent z bins
        cand = [Pb[kk, r] for kk in (k - 1, k, k + 1) if 0 <= kk < K]
        best = max(cand)
        d = abs(best - pw) / pw
        worst = max(worst, d)
        assert d <= 0.03, f"peak (k={k}, r={r}) fp32 {pw:.3f} bf16 {best:.3f}: {100 * d:.2f} % > 3 %"
        # and it must still be a local maximum there in r (no frequency drift beyond the bin)
        kb = (k - 1, k, k + 1)[int(np.argmax([Pb[kk, r] if 0 <= kk < K else -1 for kk in (k - 1, k, k + 1)]))]
        lo, hi = max(0, r - 1), min(M, r + 2)
        assert Pb[kb, r] >= Pb[kb, lo:hi].max() * (1 - 0.03)
    return mean_rel, worst


# ------------------------------------------------------------------ templates
@pytest.mark.parametrize("zmax,S", [(20.0, 1024), (96.0, 2048), (200.0, 4096), (7.5, 256)])
def test_taps_and_bank_match_oracle(F, zmax, S):
    dz = 2.0 if zmax != 7.5 else 2.5
    plan = F.Plan(1 << 16, zmax, dz, S, "f64")
    taps = plan.taps()
    bank = plan.templates()
    zs = plan.z_values()
    assert np.allclose(zs, z_values(zmax, dz))
    mm = int(plan.info.halfwidth_max)
    for k, z in enumerate(zs):
        m = oracle.halfwidth(z)
        h = oracle.template_taps(z)
        assert np.abs(taps[k, mm - m: mm + m + 1] - h).max() < 2e-15
        assert np.all(taps[k, : mm - m] == 0) and np.all(taps[k, mm + m + 1:] == 0)
        H = wrapped_bank_row(h, S)
        assert np.abs(bank[k] - H).max() < 4e-15 / S * math.sqrt(2 * m + 1) + 1e-18


def test_bank_storage_rounding(F):
    p64 = F.Plan(1 << 16, 20.0, 2.0, 1024, "f64").templates()
    p32 = F.Plan(1 << 16, 20.0, 2.0, 1024, "f32").templates()
    pbf = F.Plan(1 << 16, 20.0, 2.0, 1024, "bf16").templates()
    assert np.array_equal(p32, p64.astype(np.complex64))      # rounded once from fp64
    as_f32 = (pbf.astype(np.uint32) << 16).view(np.float32)
    # RNE from fp64 agrees with RNE from the fp32 value except on double-rounding ties (none expected)
    exp_re = bf16_rne(p64.real.astype(np.float32))
    exp_im = bf16_rne(p64.imag.astype(np.float32))
    assert np.mean(as_f32[..., 0] == exp_re) > 0.9999 and np.mean(as_f32[..., 1] == exp_im) > 0.9999
    rel = np.abs(as_f32[..., 0].astype(np.float64) - p64.real) / np.abs(p64.real)
    assert rel.max() <= 2.0 ** -8 * 1.0001


# ------------------------------------------------------------------ config 1
@pytest.fixture(scope="module")
def c1():
    w = workloads.config1()
    return w, oracle.power_plane(w.spectrum, w.zmax, w.dz)


def test_config1_fp64(F, c1):
    w, exp = c1
    plan, P = gpu_plane(F, w, "f64")
    assert tuple(P.shape) == (21, 32768)
    check_fp64(P.cpu().numpy(), exp)


@pytest.mark.parametrize("algo", ["mma", "fft"])
def test_config1_fp32(F, c1, algo):
    # fp32 variant in both forms: split-operand tensor-core sum (the default) and overlap-save FFTs
    w, exp = c1
    plan, P = gpu_plane(F, w, "f32", algorithm=algo)
    assert plan.algorithm() == algo
    check_fp32(P.cpu().numpy(), exp)
    got = P.cpu().numpy()
    k, r = np.unravel_index(np.argmax(got), got.shape)
    assert z_values(20.0, 2.0)[k] == 20.0 and r == 10000      # injected tone (z=+20, r0=10000.25)


@pytest.mark.parametrize("algo", ["mma", "fft"])
def test_config1_bf16_rules(F, c1, algo):
    w, exp = c1
    planf, Pf = gpu_plane(F, w, "f32")
    planb, Pb = gpu_plane(F, w, "bf16", algorithm=algo)
    assert planb.algorithm() == algo
    n, rec = planf.peaks(Pf, THRESH)
    assert n >= 1
    mean_rel, worst = check_bf16_rules(Pb.cpu().numpy(), Pf.cpu().numpy().astype(np.float64),
                                       [(int(a), int(b), float(c)) for a, b, c in rec])
    print(f"config1 bf16: mean rel {mean_rel:.4f}, worst peak {worst:.4f}")


def test_config1_noise_free_closed_form(F):
    # P9 on the GPU: noise-free tone, peak (z=+20, r=10000) = 100 sinc^2(0.25) to 1e-3
    w = workloads.config1(noise=False)
    for prec in ("f64", "f32"):
        _, P = gpu_plane(F, w, prec)
        got = P.cpu().numpy()
        k, r = np.unravel_index(np.argmax(got), got.shape)
        assert (k, r) == (20, 10000)
        assert abs(got[k, r] - 100.0 * np.sinc(0.25) ** 2) / 81.057 < 1e-3


# ------------------------------------------------------------------ config 2
@pytest.fixture(scope="module")
def c2():
    w = workloads.config2()
    return w, oracle.power_plane(w.spectrum, w.zmax, w.dz)


@pytest.mark.parametrize("algo", ["mma", "fft"])
def test_config2_fp32_full_plane(F, c2, algo):
    w, exp = c2
    plan, P = gpu_plane(F, w, "f32", algorithm=algo)
    assert tuple(P.shape) == (97, 1 << 19) and plan.algorithm() == algo
    err, tol = check_fp32(P.cpu().numpy(), exp)
    print(f"config2 fp32/{algo} max |dP| {err:.3e} (tol {tol:.3e})")


@pytest.mark.parametrize("algo", ["mma", "fft"])
def test_config2_bf16_rules(F, c2, algo):
    w, _ = c2
    planf, Pf = gpu_plane(F, w, "f32")
    _, Pb = gpu_plane(F, w, "bf16", algorithm=algo)
    n, rec = planf.peaks(Pf, THRESH)
    assert n >= 8
    mean_rel, worst = check_bf16_rules(Pb.cpu().numpy(), Pf.cpu().numpy().astype(np.float64),
                                       [(int(a), int(b), float(c)) for a, b, c in rec])
    print(f"config2 bf16: {n} peaks, mean rel {mean_rel:.4f}, worst peak {worst:.4f}")


def test_config2_fp64_window(F, c2):
    w, exp = c2
    _, P = gpu_plane(F, w, "f64")
    got = P[:, 100000:165536].cpu().numpy()
    check_fp64(got, exp[:, 100000:165536])


# ------------------------------------------------------------------ config 3 (bench size)
def test_config3_full_size_sampled_windows(F):
    import torch
    w = workloads.config3()
    planf, Pf = gpu_plane(F, w, "f32")
    assert tuple(Pf.shape) == (97, 1 << 22)
    M = w.M
    V = int(planf.info.valid_per_seg)
    rng = np.random.default_rng(0)
    starts = [0, M - 4096, 3 * V - 2048, 1000 * V - 2048] + [int(s) for s in rng.integers(0, M - 4096, 4)]
    starts += [int(t.r0) - 2048 for t in w.injections[:20:5] if 2048 < t.r0 < M - 4096]
    assert planf.algorithm() == "mma"                   # the launch configuration bench.py times
    planfft, Pfft = gpu_plane(F, w, "f32", algorithm="fft")
    p_peak = float(Pf.max().item())
    for s in starts:
        exp = oracle.power_plane(w.spectrum, w.zmax, w.dz, s, s + 4096)
        check_fp32(Pf[:, s:s + 4096].cpu().numpy(), exp, p_peak)
        check_fp32(Pfft[:, s:s + 4096].cpu().numpy(), exp, p_peak)
    del Pfft
    # bf16 against fp32 at full size, in the launch configuration bench.py times (auto = mma), and the FFT form
    n, rec = planf.peaks(Pf, THRESH)
    assert n >= 64
    for algo in ("auto", "fft"):
        planb, Pb = gpu_plane(F, w, "bf16", algorithm=algo)
        assert planb.algorithm() == ("mma" if algo == "auto" else "fft")
        rel_mean = float(((Pb - Pf).abs() / Pf).mean().item())
        assert rel_mean <= 0.02
        Pb_h = Pb.cpu().numpy()
        worst = 0.0
        for k, r, pw in rec:
            best = max(Pb_h[kk, r] for kk in (k - 1, k, k + 1) if 0 <= kk < 97)
            worst = max(worst, abs(best - pw) / pw)
        assert worst <= 0.03
        print(f"config3 bf16/{planb.algorithm()}: {n} peaks, mean rel {rel_mean:.4f}, worst peak {worst:.4f}")
        if algo == "auto":
            # tensor-core path element by element: oracle direct sum over the SAME bf16-rounded inputs
            for s0 in starts[:6]:
                exp_b = bf16_input_plane(w, s0, s0 + 4096)
                check_mma(Pb[:, s0:s0 + 4096].cpu().numpy(), exp_b, p_peak)
        del Pb
    del Pf
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ config 4 (batched)
def test_config4_batched_sub_batch(F):
    import torch
    idx = [0, 1, 10]
    ws = [workloads.config4_series(i) for i in idx]
    w0 = ws[0]
    plan = F.Plan(w0.N, w0.zmax, w0.dz, w0.seglen, "bf16")
    planf = F.Plan(w0.N, w0.zmax, w0.dz, w0.seglen, "f32")
    X = torch.from_numpy(np.stack([w.spectrum for w in ws])).cuda()
    Pb = plan.convolve(X)
    assert tuple(Pb.shape) == (3, 97, 1 << 21)
    for b, w in enumerate(ws):
        single = plan.convolve(X[b].contiguous())
        assert torch.equal(single, Pb[b])            # batching changes nothing, bit for bit
        Pf = planf.convolve(X[b].contiguous())
        s = int(w.injections[0].r0) - 2048 if w.injections else 777777
        exp = oracle.power_plane(w.spectrum, w.zmax, w.dz, s, s + 4096)
        check_fp32(Pf[:, s:s + 4096].cpu().numpy(), exp, float(Pf.max().item()))
        assert float(((Pb[b] - Pf).abs() / Pf).mean().item()) <= 0.02
        n, rec = planf.peaks(Pf, THRESH)
        # (a 30-300x tone between template rows and bins may or may not clear the threshold)
        for k, r, pw in rec:
            best = max(float(Pb[b, kk, r].item()) for kk in (k - 1, k, k + 1) if 0 <= kk < 97)
            assert abs(best - pw) / pw <= 0.03
        del single, Pf
    del Pb
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ config 5
def test_config5_windows_all_precisions(F):
    import torch
    w = workloads.config5()
    M = w.M
    half = 1 << 15
    wins = []
    for t in w.injections:
        s = int(min(max(0, round(t.r0) - half), M - 2 * half))
        wins.append(s)
    exps = [oracle.power_plane(w.spectrum, w.zmax, w.dz, s, s + 2 * half) for s in wins]
    # fp32
    for algo in ("fft", "mma"):
        planf, Pf = gpu_plane(F, w, "f32", algorithm=algo)
        assert tuple(Pf.shape) == (201, 1 << 22) and planf.algorithm() == algo
        p_peak = float(Pf.max().item())
        for s, exp in zip(wins, exps):
            check_fp32(Pf[:, s:s + 2 * half].cpu().numpy(), exp, p_peak)
    # bf16 against fp32
    _, Pb = gpu_plane(F, w, "bf16")
    for s in wins:
        a = Pf[:, s:s + 2 * half].cpu().numpy().astype(np.float64)
        b = Pb[:, s:s + 2 * half].cpu().numpy()
        pk = [(k, r, a[k, r]) for k, r in zip(*np.nonzero(a > THRESH))
              if a[k, r] >= a[max(0, k - 1):k + 2, max(0, r - 1):r + 2].max()]
        check_bf16_rules(b, a, pk)
    del Pb, Pf
    torch.cuda.empty_cache()
    # fp64 gold
    _, Pd = gpu_plane(F, w, "f64")
    nbad, worst, nbins = 0, 0.0, 0
    for s, exp in zip(wins, exps):
        got = Pd[:, s:s + 2 * half].cpu().numpy()
        rel = np.abs(got - exp) / exp
        nbad += int(np.count_nonzero(rel > 1e-10))
        worst = max(worst, float(rel.max()))
        nbins += rel.size
    print(f"config5 fp64: {nbad} of {nbins} bins above 1e-10, worst {worst:.3e}")
    assert nbad == 0


# ------------------------------------------------------------------ edge cases / invariants
@pytest.mark.parametrize("S,N,zmax", [(256, 2 * 1501, 8.0), (512, 2 * 4099, 20.0), (1024, 2 * 2048, 96.0),
                                      (2048, 2 * 5000, 20.0), (4096, 2 * 8191, 96.0),
                                      # M % 4 == 0: the fp32 variant runs its tensor-core form (ragged last tile)
                                      (256, 2 * 1500, 8.0), (2048, 2 * 5004, 20.0), (4096, 2 * 8192, 96.0)])
@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_ragged_and_odd_sizes(F, S, N, zmax, prec):
    # M odd / not a multiple of V / fewer than two segments; every supported segment length
    w = workloads.noise_only(N, seed=S + 1, zmax=zmax, dz=2.0, seglen=S)
    exp = oracle.power_plane(w.spectrum, zmax, 2.0)
    _, P = gpu_plane(F, w, prec)
    got = P.cpu().numpy()
    assert got.shape == exp.shape
    if prec == "f64":
        check_fp64(got, exp)
    else:
        check_fp32(got, exp)


def test_deterministic_and_shift_invariant(F):
    import torch
    w = workloads.config2()
    plan, P1 = gpu_plane(F, w, "f32")
    x = torch.from_numpy(w.spectrum).cuda()
    P2 = plan.convolve(x)
    assert torch.equal(P1, P2)                                    # bit-reproducible
    d = 333                                                        # not a multiple of V
    xs = torch.zeros_like(x)
    xs[d:] = x[:-d]
    P3 = plan.convolve(xs)
    a = P1[:, 1000:200000]
    b = P3[:, 1000 + d:200000 + d]
    assert float((a - b).abs().max().item()) <= 1e-5 * float(a.max().item()) + 1e-5   # P8


def test_zero_drift_row_is_the_power_spectrum(F):
    w = workloads.config1()
    _, P = gpu_plane(F, w, "f64")
    X = w.spectrum.astype(np.complex128)
    row = P[10].cpu().numpy()                                      # z = 0
    assert np.abs(row - (X.real ** 2 + X.imag ** 2)).max() < 1e-12 * row.max()


@pytest.mark.parametrize("prec,algo", [("f64", "fft"), ("f32", "fft"), ("f32", "mma"), ("bf16", "fft"), ("bf16", "mma")])
@pytest.mark.parametrize("zmax,dz", [(0.0, 2.0), (2.0, 2.0), (1.0, 2.0)])
def test_degenerate_banks(F, prec, algo, zmax, dz):
    # smallest banks: zmax = 0 (K = 1, the z = 0 template alone: the plane IS the power spectrum, pin P2),
    # K = 3, and zmax < dz (K = 1 at z = -1: asymmetric grid without a z = 0 row)
    import torch
    w = workloads.noise_only(1 << 14, seed=77, zmax=zmax, dz=dz, seglen=256)
    plan, P = gpu_plane(F, w, prec, algorithm=algo)
    assert plan.algorithm() == algo and P.shape[0] == (3 if zmax == 2.0 else 1)
    exp = oracle.power_plane(w.spectrum, zmax, dz)
    got = P.cpu().numpy().astype(np.float64)
    if prec == "f64":
        check_fp64(got, exp)
    elif prec == "f32":
        check_fp32(got, exp)
    else:
        assert float((np.abs(got - exp) / exp).mean()) <= 0.02
    if zmax == 0.0 and prec != "bf16":
        X = w.spectrum.astype(np.complex128)
        tol = 1e-12 if prec == "f64" else 1e-5
        assert np.abs(got[0] - (X.real ** 2 + X.imag ** 2)).max() <= tol * got.max()


# ------------------------------------------------------------------ tensor-core (MMA) path of the bf16 variant
def test_mma_config1_element_by_element(F):
    w = workloads.config1()
    plan, P = gpu_plane(F, w, "bf16")
    assert plan.algorithm() == "mma"                    # AUTO picks the tensor-core path for bf16
    err, tol = check_mma(P.cpu().numpy(), bf16_input_plane(w))
    print(f"config1 mma vs bf16-input oracle: max |dP| {err:.3e} (tol {tol:.3e})")
    got = P.cpu().numpy()
    k, r = np.unravel_index(np.argmax(got), got.shape)
    assert (k, r) == (20, 10000)                        # injected tone (z=+20, r0=10000.25)


@pytest.mark.parametrize("N,zmax,dz,S", [
    (2 * 5000, 5.0, 2.0, 1024),        # asymmetric grid z = -5..3 (no +-z pairs), M not a multiple of 128
    (2 * 70001, 200.0, 2.0, 4096),     # K = 201 -> two template groups; odd M
    (2 * 1501, 8.0, 2.0, 256),         # tiny: a few tiles, last one ragged
    (2 * 33000, 7.5, 2.5, 1024),       # fractional z step
    (2 * 4099, 96.0, 2.0, 2048),       # bench bank on a short, odd spectrum
    # M % 4 == 0: the bulk-copy kernel (staged 512-byte row segments), ragged last tile
    (2 * 5004, 5.0, 2.0, 1024),        # asymmetric grid, every entry has one plane row only
    (2 * 70004, 200.0, 2.0, 4096),     # two template groups, 15 K-steps
    (2 * 1500, 8.0, 2.0, 256),         # tiny
    (2 * 4100, 96.0, 2.0, 2048),       # bench bank, last tile of 4 bins
    (2 * 16384, 30.0, 2.0, 512),       # M a multiple of the tile; few |z| entries (empty column groups)
])
def test_mma_ragged_odd_and_grouped(F, N, zmax, dz, S):
    import torch
    w = workloads.noise_only(N, seed=S + 11, zmax=zmax, dz=dz, seglen=S)
    plan, P = gpu_plane(F, w, "bf16", algorithm="mma")
    assert plan.algorithm() == ("mma" if (N // 2) % 4 == 0 else "mma_scalar")
    got = P.cpu().numpy()
    exp = bf16_input_plane(w)
    assert got.shape == exp.shape
    check_mma(got, exp)
    # the two store paths of the tensor-core kernel hold the same bits
    plans, Ps = gpu_plane(F, w, "bf16", algorithm="mma_scalar")
    assert plans.algorithm() == "mma_scalar"
    assert torch.equal(P, Ps)
    # and the FFT form of the bf16 variant obeys the bf16 rule on the same input
    _, Pfft = gpu_plane(F, w, "bf16", algorithm="fft")
    _, Pf = gpu_plane(F, w, "f32")
    assert float(((Pfft - Pf).abs() / Pf).mean().item()) <= 0.02
    assert float(((P - Pf).abs() / Pf).mean().item()) <= 0.02


def test_mma_tap_matrix_is_the_rounded_oracle_taps(F):
    # PAPER.md:105 "converted to bfloat16": RNE once from fp64; Table 1 statistics
    for zmax, dz, S in ((96.0, 2.0, 2048), (5.0, 2.0, 1024)):
        plan = F.Plan(1 << 16, zmax, dz, S, "bf16")
        tm = plan.tapmatrix()
        mm = int(plan.info.halfwidth_max)
        rels = []
        for k, z in enumerate(plan.z_values()):
            h = oracle.template_taps(z)
            m = (len(h) - 1) // 2
            got = (tm[k].astype(np.uint32) << 16).view(np.float32)
            assert np.all(got[: mm - m] == 0) and np.all(got[mm + m + 1:] == 0)
            g = got[mm - m: mm + m + 1]
            for part, e64 in ((0, h.real), (1, h.imag)):
                big = np.abs(e64) > 1e-12                  # (z = 0: off-centre taps are quadrature noise)
                if not big.any():
                    continue
                e = bf16_rne(e64.astype(np.float32))
                assert np.mean(g[big, part] == e[big]) > 0.999      # double-rounding ties only
                rel = (g[big, part].astype(np.float64) - e64[big]) / e64[big]
                assert np.abs(rel).max() <= 2.0 ** -8 * 1.0001
                rels.append(rel)
        rels = np.concatenate(rels) * 100.0
        assert abs(rels.mean()) < 0.02 and 0.13 < rels.std() < 0.19    # paper: mean ~ -0.001 %, sigma 0.153 %


def test_mma_deterministic_batched_and_algorithm_switch(F):
    import torch
    w = workloads.noise_only(1 << 18, seed=5, zmax=96.0, dz=2.0, seglen=2048)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16")
    x = torch.from_numpy(w.spectrum).cuda()
    P1 = plan.convolve(x)
    P2 = plan.convolve(x)
    assert torch.equal(P1, P2)                                       # bit-reproducible
    xb = torch.stack([x, torch.roll(x, 17), x])
    Pb = plan.convolve(xb)
    assert torch.equal(Pb[0], P1) and torch.equal(Pb[2], P1)
    # switching the algorithm on a live plan
    assert F.fdas_set_algorithm(plan._h, F.FDAS_ALGO_FFT) == 0 and plan.algorithm() == "fft"
    Pfft = plan.convolve(x)
    assert not torch.equal(Pfft, P1)
    assert float(((Pfft - P1).abs() / P1).mean().item()) < 0.03
    assert F.fdas_set_algorithm(plan._h, F.FDAS_ALGO_AUTO) == 0 and plan.algorithm() == "mma"
    assert F.fdas_set_algorithm(plan._h, 7) == F.FDAS_ERR_INVALID_ARG
    # fp32: the split-operand tensor-core form is the default where the plane rows are 16-byte aligned
    planf = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    assert planf.algorithm() == "mma"
    assert F.fdas_set_algorithm(planf._h, F.FDAS_ALGO_MMA_SCALAR) == F.FDAS_ERR_UNSUPPORTED
    assert F.fdas_set_algorithm(planf._h, F.FDAS_ALGO_FFT) == 0 and planf.algorithm() == "fft"
    assert F.fdas_set_algorithm(planf._h, F.FDAS_ALGO_MMA) == 0 and planf.algorithm() == "mma"
    assert F.fdas_tapmatrix_host(planf._h, 0, 0) == F.FDAS_ERR_INVALID_ARG
    podd = F.Plan(2 * 4099, 20.0, 2.0, 1024, "f32")                 # odd M: FFT kernel
    assert podd.algorithm() == "fft" and F.fdas_set_algorithm(podd._h, F.FDAS_ALGO_MMA) == F.FDAS_ERR_UNSUPPORTED
    pd = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f64")
    assert pd.algorithm() == "fft" and F.fdas_set_algorithm(pd._h, F.FDAS_ALGO_MMA) == F.FDAS_ERR_UNSUPPORTED


def test_mma_zero_input_and_shift_invariance(F):
    import torch
    w = workloads.config2()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16")
    x = torch.from_numpy(w.spectrum).cuda()
    P0 = plan.convolve(torch.zeros_like(x))
    assert float(P0.abs().max().item()) == 0.0
    P1 = plan.convolve(x)
    d = 333
    xs = torch.zeros_like(x)
    xs[d:] = x[:-d]
    P3 = plan.convolve(xs)
    a = P1[:, 1000:200000]
    b = P3[:, 1000 + d:200000 + d]
    assert float((a - b).abs().max().item()) <= 1e-5 * float(a.max().item()) + 1e-5   # P8: no tile seams


# ------------------------------------------------------------------ peaks
def test_peaks_match_oracle_rule_on_gpu_plane(F):
    import torch
    w = workloads.config2()
    plan, P = gpu_plane(F, w, "f32")
    for thr in (THRESH, 12.0):
        n, rec = plan.peaks(P, thr)
        n_o, rec_o = oracle.peaks(P.cpu().numpy().astype(np.float64), thr)
        assert n == n_o == len(rec)
        assert sorted((int(a), int(b)) for a, b, _ in rec) == sorted((k, r) for k, r, _ in rec_o)
        got = {(int(a), int(b)): float(c) for a, b, c in rec}
        for k, r, v in rec_o:
            assert got[(k, r)] == np.float32(v)
    # capacity overflow follows the snprintf convention
    n2, rec2 = plan.peaks(P, 12.0, capacity=5)
    assert n2 == n and len(rec2) == 5
    n3, rec3 = plan.peaks(P, 12.0, capacity=0)
    assert n3 == n and len(rec3) == 0


@pytest.mark.parametrize("prec", ["bf16", "f32"])
def test_fused_search_equals_convolve_then_peaks(F, prec):
    # fdas_search (threshold test fused into the tensor-core epilogue for bf16) returns the plane of
    # fdas_convolve and the peak set of fdas_peaks; a candidate-buffer overflow falls back to a full scan
    import torch
    w = workloads.config2()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
    x = torch.from_numpy(w.spectrum).cuda()
    P = plan.convolve(x)
    for thr in (THRESH, 12.0, 6.0):
        n_ref, rec_ref = plan.peaks(P, thr, capacity=1 << 20)
        P2, n, rec = plan.search(x, thr, capacity=1 << 20)
        assert torch.equal(P2, P)
        assert n == n_ref == len(rec)
        assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))
    # repeated calls alternate the two candidate counters
    for _ in range(3):
        _, n, rec = plan.search(x, THRESH)
        assert n == plan.peaks(P, THRESH)[0]
    # overflow of the candidate buffer (threshold inside the noise) -> same answer through the full scan
    w2 = workloads.noise_only(1 << 19, seed=9, zmax=96.0, dz=2.0, seglen=2048)
    plan2 = F.Plan(w2.N, w2.zmax, w2.dz, w2.seglen, prec)
    x2 = torch.from_numpy(w2.spectrum).cuda()
    P2 = plan2.convolve(x2)
    n_ref, rec_ref = plan2.peaks(P2, 2.0, capacity=1 << 22)
    _, n, rec = plan2.search(x2, 2.0, capacity=1 << 22)
    assert n == n_ref and n > (1 << 18) // 4
    assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))
    # snprintf convention
    _, n3, rec3 = plan2.search(x2, 2.0, capacity=7)
    assert n3 == n_ref and len(rec3) == 7


def test_fused_search_asymmetric_grid_and_groups(F):
    import torch
    for N, zmax, dz, S in ((2 * 50001, 5.0, 2.0, 1024), (2 * 70001, 200.0, 2.0, 4096)):
        w = workloads.noise_only(N, seed=21, zmax=zmax, dz=dz, seglen=S)
        plan = F.Plan(w.N, zmax, dz, S, "bf16")
        x = torch.from_numpy(w.spectrum).cuda()
        P = plan.convolve(x)
        n_ref, rec_ref = plan.peaks(P, 7.0, capacity=1 << 20)
        P2, n, rec = plan.search(x, 7.0, capacity=1 << 20)
        assert torch.equal(P2, P) and n == n_ref and n > 10
        assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))


def test_peaks_hand_built_planes(F):
    import torch
    plan = F.Plan(2 * 1024, 4.0, 2.0, 256, "f32")     # K = 5, M = 1024
    P = torch.zeros((5, 1024), dtype=torch.float32, device="cuda")
    P[1, 2] = P[1, 3] = P[2, 2] = 4.0                  # plateau -> one peak, the lexicographically first
    P[0, 0] = 5.0                                       # corner
    P[4, 1023] = 6.0                                    # opposite corner
    P[3, 500] = 3.0
    P[4, 501] = 3.5                                     # diagonal neighbour dominates
    n, rec = plan.peaks(P, 1.0)
    assert sorted((int(a), int(b)) for a, b, _ in rec) == [(0, 0), (1, 2), (4, 501), (4, 1023)]
    n, rec = plan.peaks(P, 6.0)
    assert n == 0                                       # strictly above the threshold


def test_error_paths_on_device(F):
    import torch
    rc, h = F.fdas_plan_create(1 << 16, 20.0, 2.0, 1024, F.FDAS_F32)
    assert rc == 0
    x = torch.zeros(32768, dtype=torch.complex64, device="cuda")
    P = torch.zeros((21, 32768), dtype=torch.float32, device="cuda")
    assert F.fdas_convolve(h, x.data_ptr(), P.data_ptr()) == F.FDAS_ERR_NOT_BUILT
    assert F.fdas_build_templates(h) == 0
    assert F.fdas_convolve(h, 0, P.data_ptr()) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_convolve_batched(h, x.data_ptr(), P.data_ptr(), 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_convolve(h, x.data_ptr(), P.data_ptr()) == 0
    torch.cuda.synchronize()
    assert float(P.abs().max().item()) == 0.0          # empty input -> empty plane
    assert F.fdas_launch_count(h)[1] == 5             # taps, bank, twiddles, tap matrix (tensor-core form), convolve
    assert F.fdas_plan_destroy(h) == 0


def test_host_entry_points(F):
    import torch
    w = workloads.config1()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    x = torch.from_numpy(w.spectrum).pin_memory()
    out = torch.empty((21, 32768), dtype=torch.float32).pin_memory()
    plan.convolve_host(x, out)
    ref = plan.convolve(torch.from_numpy(w.spectrum).cuda())
    assert torch.equal(out, ref.cpu())
    rec = np.zeros(64, dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
    n = plan.search_host(w.spectrum, THRESH, rec, 64)            # pageable numpy buffers also work
    n_ref, rec_ref = plan.peaks(ref, THRESH)
    assert n == n_ref
    assert sorted(map(tuple, rec[:n].tolist())) == sorted(map(tuple, rec_ref.tolist()))
