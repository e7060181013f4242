"""GPU parity of the fp32 variant's tensor-core form (FDAS_ALGO_MMA on FDAS_F32): every operand
split into two bf16 terms, three products per tap, fp32 accumulation in TMEM.

Two bars: (i) the north_star fp32 tolerance against the plain oracle (test_gpu_parity covers it on
all configs in both forms); (ii) element by element against the oracle's direct sum of exactly
those three terms (tests/split_terms.py), to the fp32-accumulation bound of check_mma -- a wrong or
missing term shows up at the 1e-3 level, far above it."""
import numpy as np
import pytest

import oracle
from paper_2206_12205_b200 import workloads
from split_terms import split_plane
from test_gpu_parity import F, THRESH, check_fp32, check_mma, gpu_plane   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def test_config1_split_terms_element_by_element(F):
    w = workloads.config1()
    plan, P = gpu_plane(F, w, "f32", algorithm="mma")
    assert plan.algorithm() == "mma"
    err, tol = check_mma(P.cpu().numpy(), split_plane(w))
    print(f"config1 fp32/mma vs three-term oracle: max |dP| {err:.3e} (tol {tol:.3e})")


@pytest.mark.parametrize("N,zmax,dz,S", [
    (2 * 5004, 5.0, 2.0, 1024),        # asymmetric grid z = -5..3 (no +-z pairs)
    (2 * 70004, 200.0, 2.0, 4096),     # K = 201: two template groups, 15 K-steps, smallest work items
    (2 * 1500, 8.0, 2.0, 256),         # tiny, ragged last tile
    (2 * 33000, 7.5, 2.5, 1024),       # fractional z step
    (2 * 4100, 96.0, 2.0, 2048),       # bench bank, last tile of 4 bins
])
def test_f32_mma_ragged_and_grouped(F, N, zmax, dz, S):
    import torch
    w = workloads.noise_only(N, seed=S + 17, zmax=zmax, dz=dz, seglen=S)
    plan, P = gpu_plane(F, w, "f32")
    assert plan.algorithm() == "mma"
    got = P.cpu().numpy()
    check_mma(got, split_plane(w))
    check_fp32(got, oracle.power_plane(w.spectrum, zmax, dz))
    # bit-reproducible, and the FFT form agrees to the fp32 tolerance
    assert torch.equal(plan.convolve(torch.from_numpy(w.spectrum).cuda()), P)


def test_f32_batched_search_and_host_forms(F):
    import torch
    w = workloads.config2()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "f32")
    assert plan.algorithm() == "mma"
    x = torch.from_numpy(w.spectrum).cuda()
    P = plan.convolve(x)
    xb = torch.stack([x, torch.roll(x, 5), x])
    Pb = plan.convolve(xb)
    assert torch.equal(Pb[0], P) and torch.equal(Pb[2], P) and not torch.equal(Pb[1], P)
    # fused search (threshold in the epilogue) == convolve then peaks == the oracle rule on that plane
    n_ref, rec_ref = plan.peaks(P, THRESH, capacity=1 << 20)
    P2, n, rec = plan.search(x, THRESH, capacity=1 << 20)
    assert torch.equal(P2, P) and n == n_ref >= 8
    assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))
    n_o, rec_o = oracle.peaks(P.cpu().numpy().astype(np.float64), THRESH)
    assert sorted((int(a), int(b)) for a, b, _ in rec) == sorted((k, r) for k, r, _ in rec_o)
    # host-buffer form
    out = np.empty((plan.K, plan.M), dtype=np.float32)
    plan.convolve_host(np.ascontiguousarray(w.spectrum), out)
    assert np.array_equal(out, P.cpu().numpy())


@pytest.mark.parametrize("prec", ["bf16", "f32", "f64"])
def test_search_host_batched_equals_per_series_search(F, prec):
    # survey form (config 4 shape, shortened): 5 series, every other one carries a tone
    import torch
    N = 1 << 17
    specs = []
    for i in range(5):
        if i % 2 == 0:
            specs.append(workloads.harmonic_train(N, seed=100 + i, r0=3000.0 + 500 * i, z=4.0 * (i - 2), power=60.0,
                                                  rel_amplitudes=(1.0,), zmax=20.0, dz=2.0, seglen=1024).spectrum)
        else:
            specs.append(workloads.noise_only(N, seed=100 + i, zmax=20.0, dz=2.0, seglen=1024).spectrum)
    dt = np.complex128 if prec == "f64" else np.complex64
    X = np.ascontiguousarray(np.stack(specs).astype(dt))
    plan = F.Plan(N, 20.0, 2.0, 1024, prec)
    cap = 256
    peaks = np.zeros((5, cap, 3), dtype=np.int32)
    counts = np.zeros(5, dtype=np.int32)
    for rep in range(2):                                    # second call reuses the pipeline objects
        plan.search_host_batched(X, 12.0, peaks, counts, cap)
        for i in range(5):
            one = np.zeros((cap, 3), dtype=np.int32)
            n = plan.search_host(X[i], 12.0, one, cap)
            assert n == counts[i] and (n >= 1 if i % 2 == 0 else True)
            got = sorted(map(tuple, peaks[i, :min(n, cap)].tolist()))
            assert got == sorted(map(tuple, one[:min(n, cap)].tolist()))
    # the tone of series 0: r0 = 3000, z = -8 -> row (20 - 8) / 2 = 6
    rows = {(int(a), int(b)) for a, b, _ in peaks[0, :counts[0]]}
    assert (6, 3000) in rows
    assert F.fdas_search_host_batched(plan._h, X.ctypes.data, 0, 12.0, peaks.ctypes.data, cap, counts.ctypes.data) == F.FDAS_ERR_INVALID_ARG


def test_describe_convolve_counts_the_issued_tensor_work(F):
    # fdas_describe_convolve is what bench.py reads its kernel names, grids and tensor flops from: the counts must be
    # the launcher's.  Config-3 bank (49 |z| entries -> 112 columns, 129 taps -> 9 K steps): a full-width launch issues
    # tiles x 2 parts x 9 steps x 2*128*112*16 flops; a trimmed one multiplies 32, 64, 96, 112, 112, 112, 80, 48, 16
    # columns in its 9 steps (the templates that reach the step: half-width |z|/2 + 16 taps).
    import torch
    N = 1 << 20
    M = N // 2
    tiles = M // 128
    full = tiles * 2 * 9 * 2.0 * 128 * 112 * 16
    trimmed = tiles * 2 * 2.0 * 128 * 16 * (32 + 64 + 96 + 112 + 112 + 112 + 80 + 48 + 16)
    plan = F.Plan(N, 96.0, 2.0, 2048, "bf16")
    plane = torch.empty((plan.K, plan.M), dtype=torch.float32, device="cuda")
    d = plan.describe(plane)
    assert d["algorithm"] == "mma" and d["split"] == 1 and d["nch"] == 7 and d["k_steps"] == 9 and d["groups"] == 1
    assert d["kernel"] == "fdas_mma_bulk_kernel<7, float, 1>" and d["grid_y"] == 1 and 1 <= d["grid_x"] <= 1024
    assert d["tensor_flops"] == full                       # float plane, 97 templates: store-bound, every step at full width
    assert plan.describe(None)["tensor_flops"] == trimmed  # scan launch of the plane-free search
    p16 = F.Plan(N, 96.0, 2.0, 2048, "bf16", plane="bf16")
    assert p16.describe(torch.empty((p16.K, p16.M), dtype=torch.bfloat16, device="cuda"))["tensor_flops"] == trimmed
    p32 = F.Plan(N, 96.0, 2.0, 2048, "f32")
    d32 = p32.describe(plane)
    assert d32["split"] == 3 and d32["tensor_flops"] == 3 * trimmed
    # two template groups (201 templates): one grid for both, the group of narrow templates skips the K steps none of
    # its templates reaches, so the launch issues less than groups x full
    p5 = F.Plan(1 << 18, 200.0, 2.0, 4096, "f32")
    d5 = p5.describe(torch.empty((p5.K, p5.M), dtype=torch.float32, device="cuda"))
    assert d5["groups"] == 2 and d5["grid_y"] == 1 and d5["k_steps"] == 15
    assert d5["tensor_flops"] < 0.75 * 3 * 2 * ((1 << 17) // 128) * 2 * 15 * 2.0 * 128 * d5["nch"] * 16 * 16
