"""GPU parity of jerk-slab plans (fdas_plan_create_jerk, reading A25) against
oracle.power_plane_jerk, with the tolerances of the plain FDAS planes."""
import numpy as np
import pytest

import oracle
from helpers import bf16_rne, z_values
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F, THRESH, check_fp32, check_fp64, check_mma   # noqa: F401  (F is a fixture)

pytestmark = pytest.mark.gpu


def jerk_plane(F, w, jerk, prec, algo="auto"):
    import torch
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec, algorithm=algo, jerk=jerk)
    dt = np.complex128 if prec == "f64" else np.complex64
    P = plan.convolve(torch.from_numpy(np.ascontiguousarray(w.spectrum.astype(dt))).cuda())
    torch.cuda.synchronize()
    return plan, P


@pytest.mark.parametrize("jerk", [36.0, -60.0])
def test_jerk_slab_all_precisions_and_forms(F, jerk):
    w = workloads.jerk_tone(1 << 16, seed=3, r0=9000.0, z=4.0, w=36.0, power=90.0, zmax=12.0, dz=2.0, seglen=1024)
    exp = oracle.power_plane_jerk(w.spectrum, w.zmax, w.dz, jerk)
    plan, P = jerk_plane(F, w, jerk, "f64")
    assert int(plan.info.halfwidth_max) == oracle.halfwidth_jerk(12.0, jerk)
    check_fp64(P.cpu().numpy(), exp)
    for algo in ("fft", "mma"):
        plan, P = jerk_plane(F, w, jerk, "f32", algo)
        assert plan.algorithm() == algo
        check_fp32(P.cpu().numpy(), exp)
    # taps read back from the device equal the oracle's (fp64 quadrature on both sides)
    taps = plan.taps()
    m = int(plan.info.halfwidth_max)
    for k, z in enumerate(z_values(12.0, 2.0)):
        h = oracle.template_taps_jerk(float(z), jerk)
        mz = (len(h) - 1) // 2
        assert np.abs(taps[k, m - mz:m + mz + 1] - h).max() < 5e-15
        assert np.abs(taps[k, :m - mz]).max(initial=0.0) == 0.0
    # bf16 tensor-core form element by element: oracle direct sum over the bf16-rounded spectrum and taps
    X = w.spectrum
    Xb = bf16_rne(X.real).astype(np.float64) + 1j * bf16_rne(X.imag).astype(np.float64)
    rows = []
    for z in z_values(12.0, 2.0):
        h = oracle.template_taps_jerk(float(z), jerk)
        hb = bf16_rne(h.real.astype(np.float32)).astype(np.float64) + 1j * bf16_rne(h.imag.astype(np.float32)).astype(np.float64)
        rows.append(oracle.convolve_row(Xb, hb))
    planb, Pb = jerk_plane(F, w, jerk, "bf16")
    assert planb.algorithm() == "mma"
    check_mma(Pb.cpu().numpy(), np.stack(rows))
    _, Pbf = jerk_plane(F, w, jerk, "bf16", "fft")
    assert float((np.abs(Pbf.cpu().numpy() - exp) / exp).mean()) <= 0.02


# (the volume as a whole -- all slabs and the 26-neighbour peak rule in one library call -- is tested in test_gpu_volume.py)


def test_jerk_plan_errors(F):
    assert F.fdas_plan_create_jerk(1 << 16, 96.0, 2.0, float("nan"), 2048, F.FDAS_F32)[0] == F.FDAS_ERR_INVALID_ARG
    # taps too wide for the segment: m = ceil(96/2 + 1200/12) + 16 = 164 -> L = 192, V = 256 - 192 - 164 < 32
    assert F.fdas_plan_create_jerk(1 << 16, 96.0, 2.0, 1200.0, 256, F.FDAS_F32)[0] == F.FDAS_ERR_INVALID_ARG
    rc, h = F.fdas_plan_create_jerk(1 << 16, 20.0, 2.0, 0.0, 1024, F.FDAS_F32)
    assert rc == 0 and F.fdas_plan_info(h)[1].halfwidth_max == 26
    F.fdas_plan_destroy(h)
