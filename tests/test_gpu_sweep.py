"""Seeded random sweep over plan shapes (segment length, z grid, jerk, precision, form, batch, M): every
plane against the oracle with the north_star tolerances, and fdas_search against fdas_peaks."""
import numpy as np
import pytest

import oracle
from paper_2206_12205_b200 import workloads
from test_gpu_parity import F   # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def _cases(seed, n):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        S = int(rng.choice([256, 512, 1024, 2048, 4096]))
        dz = float(rng.choice([0.5, 1.0, 2.0, 2.5, 4.0]))
        zmax = float(rng.choice([0.0, 1.0, 3.0, 5.0, 8.0, 20.0, 33.0, 64.0, 96.0, 150.0]))
        jerk = float(rng.choice([0.0, 0.0, 24.0, -50.0]))
        m = int(np.ceil(zmax / 2 + abs(jerk) / 12)) + 16
        if (S - (m + 31) // 32 * 32 - m) // 32 * 32 < 32 or 2 * int(np.floor(zmax / dz + 1e-9)) + 1 > 260:
            continue
        out.append((S, dz, zmax, jerk, int(rng.integers(S, 20000)), str(rng.choice(["f32", "bf16", "f64"])),
                    str(rng.choice(["auto", "fft"])), int(rng.choice([1, 1, 3]))))
    return out


@pytest.mark.parametrize("S,dz,zmax,jerk,M,prec,algo,batch", _cases(2024, 24))
def test_random_plan_shapes(F, S, dz, zmax, jerk, M, prec, algo, batch):
    import torch
    w = workloads.noise_only(2 * M, seed=M, zmax=zmax, dz=dz, seglen=S)
    plan = F.Plan(2 * M, zmax, dz, S, prec, algorithm=algo, jerk=jerk)
    x = torch.from_numpy(w.spectrum.astype(np.complex128 if prec == "f64" else np.complex64)).cuda()
    P = plan.convolve(x if batch == 1 else torch.stack([x] * batch))
    got = (P if batch == 1 else P[batch - 1]).cpu().numpy().astype(np.float64)
    exp = oracle.power_plane_jerk(w.spectrum, zmax, dz, jerk)
    err = np.abs(got - exp)
    if prec == "f64":
        assert (err / exp).max() <= 1e-10
    elif prec == "f32":
        assert err.max() <= 1e-4 * exp.max() + 1e-4
    else:
        assert (err / exp).mean() <= 0.02
    if batch == 1 and prec != "f64":
        n_ref, rec_ref = plan.peaks(P, 6.0, capacity=1 << 18)
        P2, n, rec = plan.search(x, 6.0, capacity=1 << 18)
        assert torch.equal(P2, P) and n == n_ref
        assert sorted(map(tuple, rec.tolist())) == sorted(map(tuple, rec_ref.tolist()))
        if plan.algorithm() != "fft":                   # plane-free form: the same peak set without a plane
            _, n3, rec3 = plan.search(x, 6.0, capacity=1 << 18, plane_free=True)
            assert n3 == n_ref
            assert sorted(map(tuple, rec3.tolist())) == sorted(map(tuple, rec_ref.tolist()))
