#!/usr/bin/env python
"""bench.py -- FDAS convolution hot path on B200: plane points/s and HBM roofline fraction.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole hot path over one
spectrum of BASELINE.json config 3 (N = 2^23 samples, 97 templates, segment 2048) through the
C ABI of libfdas: fdas_search = the convolution (spectrum load, template filter bank, |.|^2,
plane store) and the threshold / local-maximum peak pass.  Headline variant: bf16 storage /
fp32 accumulate with a float plane (the north_star target; tensor-core kernel with the threshold
test fused into its epilogue).  Timed in the same run and reported under "precisions": the fp32
variant in its tensor-core form (split operands) and its overlap-save FFT form, the FFT form of
the bf16 variant, and the bf16-stored plane with the paper's quick cast.  Prints ONE JSON line
(rank 0).

N > 1: the path shards by independent series (no data-path collective):
every rank convolves its own config-3-shaped series -> weak scaling.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np

METRIC = "fdas_plane_points_per_s"
UNIT = "points/s"
THRESH = 22.5              # DESIGN.md reading A13
PEAK_CAPACITY = 1 << 16
WORKLOAD = "config3: N=2^23 fp32 samples (noise seed 3 + 64 five-harmonic pulse trains), M=2^22 bins, K=97 templates (z in [-96,96] step 2), seglen 2048 -> 97 x 2^22 plane"
N_SAMPLES = 1 << 23
ZMAX, DZ, SEGLEN = 96.0, 2.0, 2048


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)", {}


def algorithmic_bytes(K, M, S, V, plane_elem=4, spec_elem=8):
    """plane write K*M*4 B + spectrum read n_seg*S*8 B (halo re-read included)."""
    n_seg = -(-M // V)
    return K * M * plane_elem + n_seg * S * spec_elem


def hsum_bytes(K, M, H, elem=4):
    """Elements the harmonic sum must read (rows k0 + h (k - k0) in range, bins h r < M) plus the plane it writes."""
    k0 = (K - 1) // 2
    reads = sum((2 * (k0 // h) + 1) * (-(-M // h)) for h in range(1, H + 1))
    return elem * (reads + K * M)


def split_mma_columns(zmax, dz):
    """Columns each 16-tap K step of the fp32 tensor-core form multiplies (one template group, symmetric grid):
    templates whose taps do not reach a K step are skipped (fdas_mma.cu).  Accounting only."""
    m_max = int(math.ceil(zmax / 2)) + 16
    KS = -(-(2 * m_max + 1) // 16)
    nz = int(math.floor(zmax / dz + 1e-9)) + 1
    NT = -(-2 * nz // 16) * 16
    cols = []
    for ks in range(KS):
        jhi = m_max - 16 * ks
        jlo = jhi - 15
        minabs = 0 if jlo <= 0 <= jhi else min(abs(jlo), abs(jhi))
        need = sum(1 for e in range(nz) if int(math.ceil((zmax - e * dz) / 2)) + 16 >= minabs)
        cols.append(min(NT, max(16, -(-4 * ((need + 1) // 2) // 16) * 16)))
    return cols


def nominal_flops(K, M, S, V):
    """per segment 5 S log2 S (forward) + K (6S + 5 S log2 S + 3V)."""
    n_seg = -(-M // V)
    l2 = math.log2(S)
    return n_seg * (5 * S * l2 + K * (6 * S + 5 * S * l2 + 3 * V))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, reasons, mx = [], set(), None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx = float(r[2])
            except ValueError:
                continue
            for nm, v in zip(names, r[5:9]):
                if v.strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm))
        return out


def time_oracle_sample(spectrum, window_bins: int):
    """The oracle as it stands on the host cores: direct-sum rows for all K templates over a
    window of `window_bins` bins of the workload's spectrum (taps precomputed, like the GPU's
    one-off template build).  Returns (points/s, seconds, cores, description)."""
    import oracle
    zs = -ZMAX + DZ * np.arange(2 * int(ZMAX / DZ) + 1)
    taps = [oracle.template_taps(float(z)) for z in zs]
    M = len(spectrum)
    r0 = M // 2 - window_bins // 2
    X = spectrum.astype(np.complex128)
    t0 = time.perf_counter()
    for h in taps:
        oracle.convolve_row(X, h, r0, r0 + window_bins)
    dt = time.perf_counter() - t0
    pts = len(zs) * window_bins
    return pts / dt, dt, oracle.num_threads(), (
        f"oracle direct sum, all {len(zs)} templates over a {window_bins}-bin window of the config-3 spectrum "
        f"({pts:.3e} of {len(zs) * M:.3e} plane points; templates precomputed)")


def run_reference(args, rank):
    """--impl reference: the CPU oracle (oracle/fdas_oracle.c) on the host cores, bounded sample per step."""
    if rank != 0:
        return
    from paper_2206_12205_b200 import workloads
    w = workloads.noise_only(N_SAMPLES, seed=3, zmax=ZMAX, dz=DZ, seglen=SEGLEN)   # same shape; values do not change the cost
    window = 1 << 17
    for _ in range(max(0, min(args.warmup, 1))):
        time_oracle_sample(w.spectrum, 1 << 12)
    vals, secs, cores, desc = [], 0.0, 1, ""
    for _ in range(args.steps):
        v, dt, cores, desc = time_oracle_sample(w.spectrum, window)
        vals.append(v)
        secs += dt
    value = float(np.mean(vals))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--noise-only", action="store_true", help="skip the (slow) signal injection; same shapes")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    from paper_2206_12205_b200 import _build, fdas, sharding, workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libfdas has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    _build.build()
    fdas.lib()

    # ---- workload (each rank its own series: independent problems, no collective)
    if args.noise_only:
        w = workloads.noise_only(N_SAMPLES, seed=3 + 1000 * rank, zmax=ZMAX, dz=DZ, seglen=SEGLEN)
    else:
        w = workloads.config3()
        if rank:
            w.spectrum = workloads.noise_only(N_SAMPLES, seed=3 + 1000 * rank).spectrum
    stream = torch.cuda.Stream()
    sptr = stream.cuda_stream
    results = {}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    peaks_dev = torch.empty(PEAK_CAPACITY * 3, dtype=torch.int32, device="cuda")
    count_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    x_dev = torch.from_numpy(w.spectrum).cuda()
    x_pin = torch.from_numpy(w.spectrum).pin_memory()
    peaks_pin = torch.empty(PEAK_CAPACITY * 3, dtype=torch.int32).pin_memory()
    sampler = None

    # (name, precision, algorithm, plane format); headline (bf16, float plane) last so the clock sample covers it
    variants = (("f32_fft", "f32", "fft", "f32"), ("f32", "f32", "auto", "f32"), ("bf16_fft", "bf16", "fft", "f32"),
                ("bf16_plane16", "bf16", "auto", "bf16"), ("bf16", "bf16", "auto", "f32"))
    for prec, pname, algo, pfmt in variants:
        plan = fdas.Plan(w.N, ZMAX, DZ, SEGLEN, pname, stream=sptr, algorithm=algo, plane=pfmt)
        K, M, S, V = plan.K, plan.M, plan.S, int(plan.info.valid_per_seg)
        plane = torch.empty((K, M), dtype=plan.plane_dtype(), device="cuda")
        h = plan._h

        def step():
            rc = fdas.fdas_search(h, x_dev.data_ptr(), plane.data_ptr(), THRESH, peaks_dev.data_ptr(), PEAK_CAPACITY,
                                  count_dev.data_ptr(), sptr)
            assert rc == 0

        def convolve_only():
            assert fdas.fdas_convolve(h, x_dev.data_ptr(), plane.data_ptr(), sptr) == 0

        with torch.cuda.stream(stream):
            for _ in range(args.warmup):
                step()
            stream.synchronize()
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()
            if prec == "bf16" and rank == 0:
                sampler = ClockSampler(local)
            l0 = plan.launch_count()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                  for _ in range(args.steps)]
            for a, c in ev:                         # the timed region: K steps of the whole hot path
                flush.zero_()                       # L2 flush between timed iterations (untimed)
                a.record(stream)
                step()
                c.record(stream)
            stream.synchronize()
            torch.cuda.synchronize()
            launches = plan.launch_count() - l0
            if world > 1:
                dist.barrier()
            # the dominant kernel alone (roofline): fdas_convolve, same stream, same flush
            evk = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                   for _ in range(args.steps)]
            for a, b in evk:
                flush.zero_()
                a.record(stream)
                convolve_only()
                b.record(stream)
            stream.synchronize()
            cast_ms = None
            if pfmt == "bf16":                       # the paper's quick cast of the bf16-stored plane
                wide = torch.empty((K, M), dtype=torch.float32, device="cuda")
                evc = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
                for a, b in evc:
                    flush.zero_()
                    a.record(stream)
                    plan.quick_cast(plane, wide, stream=sptr)
                    b.record(stream)
                stream.synchronize()
                cast_ms = float(np.mean([a.elapsed_time(b) for a, b in evc]))
                del wide
            hsum_ms = None
            if prec == "bf16":                       # NEXT-3: harmonic sum (4 harmonics) of the headline plane
                hs = torch.empty((K, M), dtype=torch.float32, device="cuda")
                evh = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
                for a, b in evh:
                    flush.zero_()
                    a.record(stream)
                    plan.harmonic_sum(plane, 4, hs, stream=sptr)
                    b.record(stream)
                stream.synchronize()
                hsum_ms = float(np.mean([a.elapsed_time(b) for a, b in evh]))
                del hs
            rfft_ms = None
            if prec == "bf16":                       # NEXT-4: the fp32 real FFT ahead of the convolution
                ts = torch.randn(w.N, dtype=torch.float32, device="cuda")
                xo = torch.empty(M, dtype=torch.complex64, device="cuda")
                plan.spectrum(ts, xo, stream=sptr)
                evr = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
                for a, b in evr:
                    flush.zero_()
                    a.record(stream)
                    plan.spectrum(ts, xo, stream=sptr)
                    b.record(stream)
                stream.synchronize()
                rfft_ms = float(np.mean([a.elapsed_time(b) for a, b in evr]))
                del ts, xo
        conv_ms = [a.elapsed_time(b) for a, b in evk]
        step_ms = [a.elapsed_time(c) for a, c in ev]
        total_ms = sharding.max_over_ranks(float(sum(step_ms)), device="cuda")
        n_found = int(count_dev.item())

        # ---- end to end through the host-buffer entry point (H2D spectrum, convolve, peaks, D2H result)
        e2e_steps = max(3, min(args.steps, 10))
        for _ in range(2):
            n_e2e = plan.search_host(x_pin, THRESH, peaks_pin, PEAK_CAPACITY, sptr)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            n_e2e = plan.search_host(x_pin, THRESH, peaks_pin, PEAK_CAPACITY, sptr)
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
        e2e_s = sharding.max_over_ranks(e2e_s, device="cuda")
        e2e_batched_s = None
        if prec == "bf16":
            # survey form: 8 series of this shape through fdas_search_host_batched (H2D of series i+1 overlaps series i)
            nb, cap_b = 8, 4096
            xb_pin = torch.from_numpy(w.spectrum).unsqueeze(0).repeat(nb, 1).contiguous().pin_memory()
            pk_pin = torch.empty((nb, cap_b, 3), dtype=torch.int32).pin_memory()
            ct_pin = torch.zeros(nb, dtype=torch.int32).pin_memory()
            plan.search_host_batched(xb_pin, THRESH, pk_pin, ct_pin, cap_b, sptr)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(3):
                plan.search_host_batched(xb_pin, THRESH, pk_pin, ct_pin, cap_b, sptr)
            torch.cuda.synchronize()
            e2e_batched_s = sharding.max_over_ranks((time.perf_counter() - t0) / (3 * nb), device="cuda")
            del xb_pin, pk_pin, ct_pin
        results[prec] = dict(K=K, M=M, S=S, V=V, e2e_batched_s=e2e_batched_s, conv_ms=float(np.mean(conv_ms)), conv_ms_min=float(np.min(conv_ms)),
                             step_ms=total_ms / args.steps, launches=launches, n_found=n_found,
                             e2e_s=e2e_s, n_e2e=n_e2e, cast_ms=cast_ms, hsum_ms=hsum_ms, rfft_ms=rfft_ms, algorithm=plan.algorithm())
        del plane
        plan.close()

    clocks = sampler.stop() if sampler else {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    r = results["bf16"]
    rf = results["f32"]
    rff = results["f32_fft"]
    rb = results["bf16_fft"]
    rp = results["bf16_plane16"]
    K, M, S, V = r["K"], r["M"], r["S"], r["V"]
    points = K * M
    value = world * points / (r["step_ms"] * 1e-3)
    peak_gbs, peak_src, peaks_json = measured_peaks()
    alg_bytes = algorithmic_bytes(K, M, S, V)
    achieved = alg_bytes / (r["conv_ms"] * 1e-3) / 1e9
    flops = nominal_flops(K, M, S, V)
    sm_max = float(peaks_json.get("sm_max_mhz", 1965.0))
    alu_peak = 148 * 128 * 2 * sm_max * 1e6 / 1e12       # TFLOP/s fp32 FMA, DESIGN.md section 7
    # tensor-core work the MMA kernel issues: per 128-bin tile 2 parts x KS K-steps of
    # a 128 x NT x 16 MMA, NT = 16*ceil(2*49/16) = 112, KS = ceil(129/16) = 9
    nz = (K + 1) // 2
    NT = -(-2 * nz // 16) * 16
    KS = -(-(2 * (int(math.ceil(ZMAX / 2)) + 16) + 1) // 16)
    mma_flops = (-(-M // 128)) * 2 * KS * 2 * 128 * NT * 16
    split_flops = (-(-M // 128)) * 2 * 3 * sum(2 * 128 * c * 16 for c in split_mma_columns(ZMAX, DZ))
    tensor_peak = float(peaks_json.get("bf16_tflops", 1590.0))
    tensor_src = "measured (MEASURED_PEAKS.json bf16_tflops, burst)" if "bf16_tflops" in peaks_json else "fallback 1.59 PFLOP/s"
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")       # ncu dram__bytes_read.sum + dram__bytes_write.sum per launch
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["key"] == "bf16_conv":
                traffic = float(row["dram_bytes_per_launch"])

    cpu = None
    if not args.no_cpu_baseline:
        v, dt, cores, desc = time_oracle_sample(w.spectrum, 1 << 22)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": r["step_ms"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": WORKLOAD,
                   "storage": "bf16 spectrum and taps (RNE), fp32 accumulate on the tensor cores (tcgen05), fp32 plane",
                   "step": "fdas_search = convolve + threshold/local-max peaks (threshold %.1f)" % THRESH,
                   "sharding": "independent series per rank",
                   "l2": "256 MB buffer written between timed steps; plane 1.63 GB per step >> 126 MB L2",
                   "noise_only": bool(args.noise_only)},
        "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"]},
        "e2e": {"value": world * points / r["e2e_s"], "unit": UNIT,
                "h2d_bytes_per_step": int(M * 8), "d2h_bytes_per_step": int(4 + 12 * min(r["n_e2e"], PEAK_CAPACITY)),
                "api": "fdas_search_host (pinned host spectrum in, peak list out)", "ms_per_step": r["e2e_s"] * 1e3},
        "e2e_batched": {"value": world * points / r["e2e_batched_s"], "unit": UNIT, "ms_per_series": r["e2e_batched_s"] * 1e3,
                        "series_per_call": 8, "h2d_bytes_per_series": int(M * 8), "d2h_bytes_per_series": 4 + 12 * 4096,
                        "api": "fdas_search_host_batched (8 pinned host spectra per call; copy of series i+1 overlaps the search of series i)"},
        "gpu_launches": int(r["launches"]),
        "roofline": {"bound": "hbm", "kernel": "fdas_mma_bulk_kernel<7, float, 1> (fdas_convolve, bf16)", "achieved": achieved,
                     "peak": peak_gbs, "unit": "GB/s", "frac": achieved / peak_gbs, "traffic": traffic,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                     "kernel_ms": r["conv_ms"], "kernel_ms_min": r["conv_ms_min"],
                     "frac_of_nominal_8TBs": achieved / 8000.0},
        "roofline_tensor": {"bound": "tensor", "kernel": "fdas_mma_bulk_kernel<7, float, 1>", "achieved": mma_flops / (r["conv_ms"] * 1e-3) / 1e12,
                            "peak": tensor_peak, "unit": "TFLOP/s", "frac": mma_flops / (r["conv_ms"] * 1e-3) / 1e12 / tensor_peak,
                            "flops_per_launch": mma_flops, "peak_source": tensor_src,
                            "count": "issued dense MMA flops: tiles x 2 parts x 9 K-steps x 2*128*112*16 (padding included)"},
        "roofline_tensor_fp32": {"bound": "tensor", "kernel": "fdas_mma_bulk_kernel<7,float,3> (fdas_convolve, fp32 variant: bf16 x 3 split operands)",
                                 "achieved": split_flops / (rf["conv_ms"] * 1e-3) / 1e12, "peak": tensor_peak, "unit": "TFLOP/s",
                                 "frac": split_flops / (rf["conv_ms"] * 1e-3) / 1e12 / tensor_peak, "flops_per_launch": split_flops,
                                 "peak_source": tensor_src,
                                 "count": "issued dense MMA flops: 3 products per tap, columns per K step " + str(split_mma_columns(ZMAX, DZ))},
        "roofline_alu_fp32_fft": {"bound": "alu", "kernel": "fdas_convolve_kernel<TraitsF32,2048>",
                                  "achieved": flops / (rff["conv_ms"] * 1e-3) / 1e12, "peak": alu_peak,
                                  "unit": "TFLOP/s", "frac": flops / (rff["conv_ms"] * 1e-3) / 1e12 / alu_peak,
                                  "flops_per_launch": flops, "count": "nominal 5 N log2 N (SURVEY.md 8(d))"},
        "cpu_baseline": cpu,
        "precisions": {
            "bf16": {"algorithm": r["algorithm"], "convolve_ms": r["conv_ms"], "step_ms": r["step_ms"],
                     "points_per_s": points / (r["step_ms"] * 1e-3),
                     "convolve_points_per_s": points / (r["conv_ms"] * 1e-3), "hbm_gbs": achieved, "peaks_found": r["n_found"]},
            "f32": {"algorithm": rf["algorithm"], "convolve_ms": rf["conv_ms"], "step_ms": rf["step_ms"],
                    "points_per_s": points / (rf["step_ms"] * 1e-3),
                    "convolve_points_per_s": points / (rf["conv_ms"] * 1e-3),
                    "hbm_gbs": alg_bytes / (rf["conv_ms"] * 1e-3) / 1e9, "peaks_found": rf["n_found"],
                    "note": "FDAS_ALGO_MMA on FDAS_F32: operands split into two bf16 terms, three products per tap"},
            "f32_fft": {"algorithm": rff["algorithm"], "convolve_ms": rff["conv_ms"], "step_ms": rff["step_ms"],
                        "points_per_s": points / (rff["step_ms"] * 1e-3),
                        "convolve_points_per_s": points / (rff["conv_ms"] * 1e-3),
                        "hbm_gbs": alg_bytes / (rff["conv_ms"] * 1e-3) / 1e9, "peaks_found": rff["n_found"],
                        "note": "FDAS_ALGO_FFT: the overlap-save FFT kernel (PAPER.md:65-67) + separate peak pass"},
            "bf16_fft": {"algorithm": rb["algorithm"], "convolve_ms": rb["conv_ms"], "step_ms": rb["step_ms"],
                         "points_per_s": points / (rb["step_ms"] * 1e-3),
                         "convolve_points_per_s": points / (rb["conv_ms"] * 1e-3),
                         "hbm_gbs": alg_bytes / (rb["conv_ms"] * 1e-3) / 1e9, "peaks_found": rb["n_found"],
                         "note": "FDAS_ALGO_FFT: the overlap-save FFT kernel with bf16 storage"},
            "bf16_plane16": {"algorithm": rp["algorithm"], "convolve_ms": rp["conv_ms"], "step_ms": rp["step_ms"],
                             "quick_cast_ms": rp["cast_ms"], "points_per_s": points / (rp["step_ms"] * 1e-3),
                             "convolve_points_per_s": points / (rp["conv_ms"] * 1e-3),
                             "hbm_gbs": algorithmic_bytes(K, M, S, V, plane_elem=2) / (rp["conv_ms"] * 1e-3) / 1e9,
                             "quick_cast_hbm_gbs": None if not rp["cast_ms"] else 6.0 * points / (rp["cast_ms"] * 1e-3) / 1e9,
                             "peaks_found": rp["n_found"],
                             "note": "NEXT-1: bf16-stored plane (PAPER.md:91-93) + fdas_quick_cast timed separately"},
            "harmonic_sum_4": {"ms": r["hsum_ms"],
                               "algorithmic_gbs": None if not r["hsum_ms"] else hsum_bytes(K, M, 4) / (r["hsum_ms"] * 1e-3) / 1e9,
                               "note": "NEXT-3: fdas_harmonic_sum, 4 harmonics, on the headline float plane; bytes = elements read + plane written"},
            "real_fft": {"ms": r["rfft_ms"], "algorithmic_gbs": None if not r["rfft_ms"] else 6.0 * 4 * M / (r["rfft_ms"] * 1e-3) / 1e9,
                         "note": "NEXT-4: fdas_spectrum, fp32 real FFT of the 2^23-sample series (outside the timed step, as in the paper); "
                                 "bytes = series read + spectrum written (3 passes move 3x that)"},
            "bf16_over_fp32_speedup": rf["conv_ms"] / r["conv_ms"],
            "bf16_over_fp32_speedup_whole_step": rf["step_ms"] / r["step_ms"],
            "bf16_over_fp32_fft_speedup": rff["conv_ms"] / r["conv_ms"],
            "bf16_fft_over_fp32_fft_speedup": rff["conv_ms"] / rb["conv_ms"],
            "paper_bf16_over_fp32_speedup": "~1.6x on 'NVIDIA Ampere' (PAPER.md:15; context, not the target)",
        },
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
