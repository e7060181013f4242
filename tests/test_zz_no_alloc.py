"""fdas_search_static (include/fdas.h): the plane-free search whose scratch is a device array compiled into the
library, for callers that cannot allocate.  Same kernels as fdas_search, so the peak set must equal the existing
paths' -- cells and power bits -- on calls in a row that share the array (different spectra, different plans), and
the entry point must refuse what does not fit the array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2206_12205_b200 import workloads

pytestmark = pytest.mark.gpu

THRESH = 22.5   # DESIGN.md reading A13


@pytest.fixture(scope="module")
def F():
    import torch
    assert torch.cuda.is_available()
    from paper_2206_12205_b200 import _build, fdas
    _build.build()
    fdas.lib()
    return fdas


def as_set(rec):
    return sorted(map(tuple, rec.tolist()))


def static_search(plan, x, thr, peaks_buf, count_buf, capacity):
    """one fdas_search_static call into caller-owned buffers -> (total, records)"""
    plan.search_static(x, thr, peaks_buf, count_buf, capacity)
    n = int(count_buf.item())
    w = min(n, capacity)
    raw = peaks_buf[: 3 * w].cpu().numpy().reshape(w, 3)
    rec = np.zeros(w, dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
    rec["z_index"] = raw[:, 0]
    rec["r"] = raw[:, 1]
    rec["power"] = raw[:, 2].copy().view(np.float32)
    return n, rec


@pytest.mark.parametrize("prec", ["bf16", "f32"])
def test_static_search_equals_the_existing_paths_on_calls_in_a_row(F, prec):
    import torch
    w = workloads.config2()                                              # 97 templates x 2^19 bins, pulses in noise
    w2 = workloads.noise_only(w.N, seed=77, zmax=w.zmax, dz=w.dz, seglen=w.seglen)
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, prec)
    xa = torch.from_numpy(w.spectrum).cuda()
    xb = torch.from_numpy(w2.spectrum).cuda()
    cap = 1 << 18
    peaks_buf = torch.empty(3 * cap, dtype=torch.int32, device="cuda")
    count_buf = torch.zeros(1, dtype=torch.int32, device="cuda")
    # two calls in a row on different inputs and thresholds, then the first again: the shared array carries nothing over
    got = [static_search(plan, x, thr, peaks_buf, count_buf, cap) for x, thr in ((xa, THRESH), (xb, 7.0), (xa, THRESH), (xa, 6.0))]
    for (n, rec), (x, thr) in zip(got, ((xa, THRESH), (xb, 7.0), (xa, THRESH), (xa, 6.0))):
        _, n_plane, rec_plane = plan.search(x, thr, capacity=cap)                      # convolve into a plane + fused peaks
        _, n_free, rec_free = plan.search(x, thr, capacity=cap, plane_free=True)       # plane-free, plan-owned scratch
        assert n == n_plane == n_free, (thr, n, n_plane, n_free)
        assert as_set(rec) == as_set(rec_plane) == as_set(rec_free)                    # bit-exact: same kernels, same arithmetic
    assert got[0][0] >= 8 and got[1][0] > 100 and as_set(got[0][1]) == as_set(got[2][1])
    # snprintf convention and capacity 0, as for fdas_search
    n7, rec7 = static_search(plan, xa, 6.0, peaks_buf, count_buf, 7)
    assert n7 == got[3][0] and len(rec7) == 7
    n0, rec0 = static_search(plan, xa, 6.0, peaks_buf, count_buf, 0)
    assert n0 == got[3][0] and len(rec0) == 0


def test_static_search_at_the_size_limit_shares_the_array_between_plans_and_allocates_nothing(F):
    import torch
    big = workloads.noise_only(1 << 23, seed=5, zmax=96.0, dz=2.0, seglen=2048)       # M = 2^22 = FDAS_SEARCH_STATIC_MAX_BINS
    assert big.N // 2 == F.FDAS_SEARCH_STATIC_MAX_BINS
    small = workloads.noise_only(2 * 70001, seed=6, zmax=20.0, dz=2.0, seglen=1024)   # odd M, ragged last tile
    p_big = F.Plan(big.N, big.zmax, big.dz, big.seglen, "bf16")
    p_small = F.Plan(small.N, small.zmax, small.dz, small.seglen, "bf16")
    x_big = torch.from_numpy(big.spectrum).cuda()
    x_small = torch.from_numpy(small.spectrum).cuda()
    cap = 1 << 16
    peaks_buf = torch.empty(3 * cap, dtype=torch.int32, device="cuda")
    count_buf = torch.zeros(1, dtype=torch.int32, device="cuda")
    ref_big = p_big.search(x_big, 9.0, capacity=cap, plane_free=True)[1:]
    ref_small = p_small.search(x_small, 5.0, capacity=cap, plane_free=True)[1:]
    # warm-up (the first launch of a kernel loads it), then two plans taking turns on the one array, memory watched
    static_search(p_big, x_big, 9.0, peaks_buf, count_buf, cap)
    static_search(p_small, x_small, 5.0, peaks_buf, count_buf, cap)
    st = torch.cuda.current_stream().cuda_stream
    peaks_2 = torch.empty(3 * cap, dtype=torch.int32, device="cuda")
    count_2 = torch.zeros(1, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    assert F.fdas_search_static(p_big._h, x_big.data_ptr(), 9.0, peaks_buf.data_ptr(), cap, count_buf.data_ptr(), st) == 0
    assert F.fdas_search_static(p_small._h, x_small.data_ptr(), 5.0, peaks_2.data_ptr(), cap, count_2.data_ptr(), st) == 0
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before                                 # no cudaMalloc happened
    for (n_ref, rec_ref), pb, cb in ((ref_big, peaks_buf, count_buf), (ref_small, peaks_2, count_2)):
        n = int(cb.item())
        assert n == n_ref and n > 10
        raw = pb[: 3 * n].cpu().numpy().reshape(n, 3)
        got = sorted((int(a), int(b), float(np.int32(c).view(np.float32))) for a, b, c in raw)
        assert got == as_set(rec_ref)


def test_static_search_refuses_what_does_not_fit(F):
    import torch
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    buf = torch.empty(3 * 16, dtype=torch.int32, device="cuda")
    # beyond the array: M = 2^23 bins
    too_big = F.Plan(1 << 24, 4.0, 2.0, 1024, "bf16")
    x = torch.zeros(too_big.M, dtype=torch.complex64, device="cuda")
    rc = F.fdas_search_static(too_big._h, x.data_ptr(), 9.0, buf.data_ptr(), 16, cnt.data_ptr(), 0)
    assert rc == F.FDAS_ERR_TOO_LARGE and F.fdas_status_string(rc) == "FDAS_ERR_TOO_LARGE"
    # two template groups (K = 201), fp64 (FFT form only): no kernel for them here
    for plan in (F.Plan(1 << 17, 200.0, 2.0, 4096, "bf16"), F.Plan(1 << 17, 20.0, 2.0, 1024, "f64")):
        xs = torch.zeros(plan.M, dtype=plan.spectrum_dtype(), device="cuda")
        assert F.fdas_search_static(plan._h, xs.data_ptr(), 9.0, buf.data_ptr(), 16, cnt.data_ptr(), 0) == F.FDAS_ERR_UNSUPPORTED
    ok = F.Plan(1 << 17, 20.0, 2.0, 1024, "bf16")
    xs = torch.zeros(ok.M, dtype=torch.complex64, device="cuda")
    assert F.fdas_search_static(ok._h, 0, 9.0, buf.data_ptr(), 16, cnt.data_ptr(), 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_search_static(ok._h, xs.data_ptr(), 9.0, 0, 16, cnt.data_ptr(), 0) == F.FDAS_ERR_INVALID_ARG
    assert F.fdas_search_static(ok._h, xs.data_ptr(), 9.0, buf.data_ptr(), 16, cnt.data_ptr(), 0) == 0
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0                                                        # an all-zero spectrum has no peak


def test_static_search_can_be_captured_into_a_cuda_graph(F):
    # what the entry point is for: stream capture rejects cudaMalloc, so a captured call proves there is none.  The
    # first call of a plan sets up function attributes and the scratch address; it is made before the capture.
    import torch
    w = workloads.config2()
    plan = F.Plan(w.N, w.zmax, w.dz, w.seglen, "bf16")
    x = torch.from_numpy(w.spectrum).cuda()
    cap = 1 << 12
    peaks_buf = torch.empty(3 * cap, dtype=torch.int32, device="cuda")
    count_buf = torch.zeros(1, dtype=torch.int32, device="cuda")
    _, n_ref, rec_ref = plan.search(x, THRESH, capacity=cap)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        assert F.fdas_search_static(plan._h, x.data_ptr(), THRESH, peaks_buf.data_ptr(), cap, count_buf.data_ptr(), s.cuda_stream) == 0
    s.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        rc = F.fdas_search_static(plan._h, x.data_ptr(), THRESH, peaks_buf.data_ptr(), cap, count_buf.data_ptr(), s.cuda_stream)
    assert rc == 0
    for _ in range(2):                                   # two replays in a row: the array is cleared inside the graph
        peaks_buf.zero_()
        count_buf.zero_()
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        n = int(count_buf.item())
        assert n == n_ref and n >= 8
        got = sorted((int(a), int(b), float(np.int32(c).view(np.float32))) for a, b, c in peaks_buf[: 3 * n].cpu().numpy().reshape(n, 3))
        assert got == as_set(rec_ref)
