"""GPU parity for the bf16-stored plane and the quick cast.

Expected values come from the oracle only: the fp64 direct sum over the bf16-rounded inputs
(test_gpu_parity.bf16_input_plane) followed by oracle.bf16 (round to nearest even, quick cast).
Bars:
  * quick cast: bit-exact (byte work);
  * bf16 plane: the stored value is the RNE rounding of the fp32 power the kernel computes, whose
    own error bound is check_mma's 1e-5 P_peak + 1e-5: so every bin must lie within half a bf16
    ulp (2^-9 relative) of the oracle power plus that bound, and must be bit-identical to the
    oracle's rounding wherever the oracle power is not within that bound of a rounding tie;
  * the north_star bf16 rules (peaks within 3 %, same or adjacent z bin; mean relative error
    <= 2 %) against the GPU fp32 plane, after the quick cast.
"""
import numpy as np
import pytest

import oracle
from oracle import bf16 as obf
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH, bf16_input_plane, check_bf16_rules, gpu_plane   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def bf16_plane_gpu(F, w, algorithm="auto"):
    import torch
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16", algorithm=algorithm, plane="bf16")
    x = torch.from_numpy(np.ascontiguousarray(w.spectrum.astype(np.complex64))).cuda()
    P = plan.convolve(x)
    torch.cuda.synchronize()
    assert P.dtype == torch.bfloat16 and int(plan.info.plane_elem_bytes) == 2
    return plan, P, x


def bits_of(P):
    import torch
    return P.view(torch.int16).cpu().numpy().view(np.uint16)


def check_bf16_plane_bits(bits, exp, p_peak=None):
    """bits: GPU plane (uint16); exp: oracle fp64 powers over the same bf16-rounded inputs."""
    if p_peak is None:
        p_peak = float(exp.max())
    tol = 1e-5 * p_peak + 1e-5                       # fp32 accumulation bound (check_mma)
    got = obf.quick_cast(bits).astype(np.float64)
    half_ulp = np.abs(exp) * 2.0 ** -8               # >= half a bf16 ulp of any value in exp's binade
    err = np.abs(got - exp)
    assert (err <= half_ulp + tol).all(), f"worst excess {(err - half_ulp - tol).max():.3e}"
    want = obf.to_bf16_bits(exp.astype(np.float32))
    differs = bits != want
    # a different pattern is legitimate only next to a rounding tie: both neighbours within tol of equidistant
    if differs.any():
        lo = obf.quick_cast(np.minimum(bits, want)[differs]).astype(np.float64)
        hi = obf.quick_cast(np.maximum(bits, want)[differs]).astype(np.float64)
        assert (np.abs(np.maximum(bits, want)[differs].astype(np.int64) - np.minimum(bits, want)[differs]) == 1).all()
        mid = 0.5 * (lo + hi)
        assert (np.abs(exp[differs] - mid) <= tol * 1.01 + 2.0 ** -24 * np.abs(exp[differs])).all()
    frac = float(differs.mean())
    assert frac < 2e-3, f"{100 * frac:.3f} % of the bins differ from the oracle rounding"
    return frac


def test_quick_cast_bit_exact_all_patterns(F):
    import torch
    # a [K][M] "plane" that holds every 16-bit pattern (NaNs and infinities included), seeded shuffle
    plan = F.Plan(2 * 8192, 20.0, 2.0, 1024, "bf16")
    K, M = plan.K, plan.M
    rng = np.random.default_rng(5)
    bits = np.resize(rng.permutation(65536).astype(np.uint16), K * M).reshape(K, M)
    src = torch.from_numpy(bits.view(np.int16)).cuda().view(torch.bfloat16)
    out = plan.quick_cast(src)
    got = out.view(torch.int32).cpu().numpy().view(np.uint32)
    want = obf.quick_cast(bits).view(np.uint32)
    assert np.array_equal(got, want)
    # batched form
    src3 = torch.stack([src, src.flip(1)])
    got3 = plan.quick_cast(src3).view(torch.int32).cpu().numpy().view(np.uint32)
    assert np.array_equal(got3[0], want) and np.array_equal(got3[1], want[:, ::-1])


def test_config1_bf16_plane_element_by_element(F):
    w = workloads.config1()
    exp = bf16_input_plane(w)
    for algo in ("mma", "mma_scalar"):
        plan, P, _ = bf16_plane_gpu(F, w, algo)
        assert plan.algorithm() == algo
        frac = check_bf16_plane_bits(bits_of(P), exp)
        print(f"config1 bf16 plane/{algo}: {100 * frac:.4f} % of bins off the oracle rounding (ties)")
    # quick cast of the GPU plane, then the north_star bf16 rules against the GPU fp32 plane
    planf, Pf = gpu_plane(F, w, "f32")
    n, rec = planf.peaks(Pf, THRESH)
    wide = plan.quick_cast(P)
    mean_rel, worst = check_bf16_rules(wide.cpu().numpy(), Pf.cpu().numpy().astype(np.float64),
                                       [(int(a), int(b), float(c)) for a, b, c in rec])
    got = wide.cpu().numpy()
    assert np.unravel_index(np.argmax(got), got.shape) == (20, 10000)     # the injected tone (z=+20, r0=10000.25)
    print(f"config1 bf16 plane: mean rel {mean_rel:.4f}, worst peak {worst:.4f}")


def test_config2_bf16_plane_rules_and_rounding_of_the_same_kernel(F):
    import torch
    w = workloads.config2()
    plan, P, x = bf16_plane_gpu(F, w)
    assert plan.algorithm() == "mma"
    planf, Pf = gpu_plane(F, w, "f32")
    n, rec = planf.peaks(Pf, THRESH)
    assert n >= 8
    wide = plan.quick_cast(P)
    mean_rel, worst = check_bf16_rules(wide.cpu().numpy(), Pf.cpu().numpy().astype(np.float64),
                                       [(int(a), int(b), float(c)) for a, b, c in rec])
    print(f"config2 bf16 plane: {n} peaks, mean rel {mean_rel:.4f}, worst peak {worst:.4f}")
    # one rounding only: the bf16 plane equals the float plane of the same kernel rounded to nearest even
    plan32, P32 = gpu_plane(F, w, "bf16", algorithm="mma")
    assert torch.equal(P32.to(torch.bfloat16).view(torch.int16), P.view(torch.int16))
    # a window around the brightest injection, element by element against the oracle
    k, r, _ = max(rec.tolist(), key=lambda t: t[2])
    s0 = max(0, int(r) - 2048)
    exp = bf16_input_plane(w, s0, s0 + 4096)
    check_bf16_plane_bits(bits_of(P[:, s0:s0 + 4096].contiguous()), exp, float(Pf.max().item()))


@pytest.mark.parametrize("N,zmax,dz,S", [
    (2 * 4099, 96.0, 2.0, 2048),       # odd M: scalar-store kernel
    (2 * 4100, 96.0, 2.0, 2048),       # M % 8 == 4: rows are not 16-byte aligned in bf16 -> scalar-store kernel
    (2 * 4104, 96.0, 2.0, 2048),       # M % 8 == 0: box stores, ragged last tile
    (2 * 70008, 200.0, 2.0, 4096),     # two template groups
    (2 * 5008, 5.0, 2.0, 1024),        # asymmetric grid (no +-z pairs)
])
def test_bf16_plane_ragged_and_grouped(F, N, zmax, dz, S):
    w = workloads.noise_only(N, seed=S + 13, zmax=zmax, dz=dz, seglen=S)
    plan, P, _ = bf16_plane_gpu(F, w)
    assert plan.algorithm() == ("mma" if (N // 2) % 8 == 0 else "mma_scalar")
    check_bf16_plane_bits(bits_of(P), bf16_input_plane(w))


def test_peaks_and_fused_search_on_a_bf16_plane(F):
    import torch
    w = workloads.config2()
    plan, P, x = bf16_plane_gpu(F, w)
    # (1) the peak kernel on a bf16 plane built by the oracle (rounding creates ties: plateau rule)
    exp_bits = obf.bf16_plane(oracle.power_plane(w.spectrum, w.zmax, w.dz).astype(np.float32))
    Pd = torch.from_numpy(exp_bits.view(np.int16)).cuda().view(torch.bfloat16)
    for thr in (THRESH, 8.0):
        n, rec = plan.peaks(Pd, thr, capacity=1 << 20)
        n_o, rec_o = oracle.peaks(obf.quick_cast(exp_bits).astype(np.float64), thr)
        assert n == n_o == len(rec)
        assert sorted((int(a), int(b), float(c)) for a, b, c in rec) == sorted((k, r, float(np.float32(v))) for k, r, v in rec_o)
    # (2) fused search == convolve then peaks, on the stored (rounded) values
    for thr in (THRESH, 8.0):
        n_ref, rec_ref = plan.peaks(P, thr, capacity=1 << 20)
        P2, n, rec = plan.search(x, thr, capacity=1 << 20)
        assert torch.equal(P2.view(torch.int16), P.view(torch.int16))
        assert n == n_ref == len(rec)
        assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))


def test_plane_format_errors_and_host_path(F):
    import torch
    w = workloads.config1()
    p32 = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    assert F.fdas_set_plane_format(p32._h, F.FDAS_PLANE_BF16) == 5          # UNSUPPORTED: not a tensor-core plan
    assert F.fdas_set_plane_format(p32._h, 7) == 1                          # INVALID_ARG
    pb = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16", plane="bf16")
    assert F.fdas_get_plane_format(pb._h) == (0, F.FDAS_PLANE_BF16)
    assert F.fdas_set_algorithm(pb._h, F.FDAS_ALGO_FFT) == 5                # the FFT kernels write float planes only
    # host-buffer form returns the same bits
    out = np.empty((pb.K, pb.M), dtype=np.uint16)
    pb.convolve_host(np.ascontiguousarray(w.spectrum.astype(np.complex64)), out)
    x = torch.from_numpy(np.ascontiguousarray(w.spectrum.astype(np.complex64))).cuda()
    assert np.array_equal(out, bits_of(pb.convolve(x)))
    # and back to float
    assert F.fdas_set_plane_format(pb._h, F.FDAS_PLANE_F32) == 0
    assert F.fdas_plan_info(pb._h)[1].plane_elem_bytes == 4


def test_config3_size_bf16_plane_sampled_windows(F):
    import torch
    w = workloads.noise_only(1 << 23, seed=3, zmax=96.0, dz=2.0, seglen=2048)   # config-3 shape (bench launch configuration)
    plan, P, _ = bf16_plane_gpu(F, w)
    assert tuple(P.shape) == (97, 1 << 22) and plan.algorithm() == "mma"
    M = w.M
    p_peak = float(P.float().max().item())
    for s0 in (0, M - 2048, 1920 * 1000 - 1024, 1234567):
        exp = bf16_input_plane(w, s0, s0 + 2048)
        check_bf16_plane_bits(bits_of(P[:, s0:s0 + 2048].contiguous()), exp, p_peak)
    del P
    torch.cuda.empty_cache()
