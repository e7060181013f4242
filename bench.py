#!/usr/bin/env python
"""bench.py -- FDAS convolution hot path on B200: plane points/s and roofline fractions.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A step = one pass of the whole hot path over one spectrum of
BASELINE.json config 3 (N = 2^23 samples, 97 templates, segment 2048) through the C ABI of libfdas:
fdas_search = the convolution (spectrum load, template filter bank, |.|^2, plane store) and the threshold /
local-maximum peak pass.  Headline variant: bf16 storage / fp32 accumulate with a float plane (the north_star
target; tensor-core kernel with the threshold test fused into its epilogue).

Timed in the same run and reported per precision (`precisions`, also under `roofline.per_precision`): the
plane-free search (no plane in HBM; tensor roofline), the bf16-stored plane with the paper's quick cast, the
fp32 variant in its split-operand tensor-core form (`f32_split3`) and in true fp32 arithmetic (`f32_fft`, the
overlap-save FFT form), the bf16 FFT form, and fp64 (the paper's "gold standard").  `configs` (also under
`roofline.per_config`) holds cold-L2 CUDA-event timings of fdas_convolve for BASELINE.json configs 1, 2, 4 and 5.
Kernel names, grids and issued tensor flops come from the library (fdas_describe_convolve), not from this file.
Prints ONE JSON line (rank 0).

N > 1: the path shards by independent series (no data-path collective): every rank
convolves its own config-3-shaped series -> weak scaling; the config-4 survey block splits its 256 series over
the ranks (paper_2206_12205_b200/sharding.py).
"""
from __future__ import annotations

import argparse
import csv
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
BAND_F_BIN = 100000.0      # fundamental of the band-maxima timing: bins 0 .. 16.5e5 of the 2^22 = 0.39 of the plane
WORKLOAD = "config3: N=2^23 fp32 samples (noise seed 3 + 64 five-harmonic pulse trains), M=2^22 bins, K=97 templates (z in [-96,96] step 2), seglen 2048 -> 97 x 2^22 plane"
N_SAMPLES = 1 << 23
ZMAX, DZ, SEGLEN = 96.0, 2.0, 2048


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)", {}


def algorithmic_bytes(K, M, S, V, plane_elem=4, spec_elem=8, batch=1):
    """plane write K*M*elem + spectrum read n_seg*S*8 B (halo re-read included), per series."""
    n_seg = -(-M // V)
    return batch * (K * M * plane_elem + n_seg * S * spec_elem)


def hsum_bytes(K, M, H, elem=4):
    """Elements the harmonic sum must read (rows k0 + h (k - k0) in range, bins h r < M) plus the plane it writes."""
    k0 = (K - 1) // 2
    reads = sum((2 * (k0 // h) + 1) * (-(-M // h)) for h in range(1, H + 1))
    return elem * (reads + K * M)


def nominal_flops(K, M, S, V, batch=1):
    """per segment 5 S log2 S (forward) + K (6S + 5 S log2 S + 3V)."""
    n_seg = -(-M // V)
    l2 = math.log2(S)
    return batch * n_seg * (5 * S * l2 + K * (6 * S + 5 * S * l2 + 3 * V))


def dram_traffic_of(kernel_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of exactly this kernel on config 3, from the committed
    ncu --set full capture (profiles/traffic.csv); None when the launcher picked a kernel no capture exists for."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tp):
        return None
    for row in csv.DictReader(open(tp)):
        if row["kernel"].replace(" ", "") == kernel_name.replace(" ", ""):
            return float(row["dram_bytes_per_launch"])
    return None


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


class Timer:
    """CUDA-event timing of calls enqueued on `stream`, a 256 MB buffer rewritten (untimed) before each call."""

    def __init__(self, torch, stream):
        self.torch, self.stream = torch, stream
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def __call__(self, fn, reps, warm=0):
        torch, st = self.torch, self.stream
        with torch.cuda.stream(st):
            for _ in range(warm):
                fn()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
            for a, b in ev:
                self.flush.zero_()
                a.record(st)
                fn()
                b.record(st)
            st.synchronize()
        return [a.elapsed_time(b) for a, b in ev]


def bench_other_configs(fdas, workloads, torch, timer, sptr, peak_gbs, tensor_peak, alu_peak, reps=10):
    """BASELINE.json configs 1, 2, 4 (one sub-batch of 32 series) and 5: fdas_convolve alone, cold L2, per precision."""
    out = {}
    # config 5 is timed BEFORE the config-4 sub-batch: for a few seconds after those 26 GB launches (about 250 GB written) the
    # same config-5 launch on the same buffers runs 5-30 % slower (0.87 ms right after, 0.78 ms a second later, 0.74 ms after
    # 3 s idle, clocks reported unchanged): a transient of the device's memory system, not of the kernel
    specs = [
        ("config1", workloads.config1(), 1, ("bf16", "f32_split3", "f32_fft", "f64"), "as BASELINE.json"),
        ("config2", workloads.config2(), 1, ("bf16", "f32_split3", "f32_fft"), "as BASELINE.json"),
        ("config5", workloads.noise_only(1 << 23, seed=4, zmax=200.0, dz=2.0, seglen=4096), 1, ("bf16", "f32_split3", "f32_fft", "f64"),
         "config-5 shape (K = 201, segment 4096) on the noise of seed 4 without the 32 tones: the time does not depend on the values"),
        ("config4_sub_batch_32", None, 32, ("bf16", "f32_split3"),
         "32 of the 256 series in one fdas_convolve_batched launch (26 GB of planes; 208 GB do not fit at once): series 0..31"),
    ]
    for name, w, batch, precs, note in specs:
        if w is None:
            ws = [workloads.config4_series(i) for i in range(batch)]
            w = ws[0]
            spec = np.stack([x.spectrum for x in ws])
        else:
            spec = w.spectrum
        entry = {"note": note, "batch": batch}
        for pn in precs:
            prec, algo = {"bf16": ("bf16", "auto"), "f32_split3": ("f32", "auto"), "f32_fft": ("f32", "fft"), "f64": ("f64", "fft")}[pn]
            plan = fdas.Plan(w.N, w.zmax, w.dz, w.seglen, prec, stream=sptr, algorithm=algo)
            K, M, S, V = plan.K, plan.M, plan.S, int(plan.info.valid_per_seg)
            x = torch.from_numpy(np.ascontiguousarray(spec.astype(np.complex128 if prec == "f64" else np.complex64))).cuda()
            shape = (K, M) if batch == 1 else (batch, K, M)
            plane = torch.empty(shape, dtype=plan.plane_dtype(), device="cuda")
            h = plan._h

            def conv():
                assert fdas.fdas_convolve_batched(h, x.data_ptr(), plane.data_ptr(), batch, sptr) == 0

            ms = timer(conv, reps, warm=3)
            info = plan.describe(plane, batch)
            elem = 8 if prec == "f64" else 4
            ab = algorithmic_bytes(K, M, S, V, plane_elem=elem, spec_elem=2 * elem, batch=batch)
            t = float(np.mean(ms)) * 1e-3
            rec = {"kernel": info["kernel"], "algorithm": info["algorithm"], "convolve_ms": float(np.mean(ms)),
                   "convolve_ms_min": float(np.min(ms)), "points_per_s": batch * K * M / t,
                   "algorithmic_bytes": ab, "hbm_gbs": ab / t / 1e9, "hbm_frac_of_measured_peak": ab / t / 1e9 / peak_gbs}
            if info["tensor_flops"] > 0:
                rec["tensor_tflops_issued"] = info["tensor_flops"] / t / 1e12
                rec["tensor_frac_of_measured_peak"] = rec["tensor_tflops_issued"] / tensor_peak
            else:
                fl = nominal_flops(K, M, S, V, batch)
                rec["alu_tflops_nominal"] = fl / t / 1e12
                rec["alu_frac"] = fl / t / 1e12 / (alu_peak if prec != "f64" else alu_peak / 2)
            entry[pn] = rec
            del plane, x
            plan.close()
            torch.cuda.empty_cache()
        entry["shape"] = {"K": K, "M": M, "S": S}
        out[name] = entry
    return out


def bench_config4_survey(fdas, workloads, sharding, torch, stream, rank, world, n_series=256):
    """BASELINE.json config 4 as a survey: all 256 series through the plane-free fdas_search_batched (no plane in HBM),
    series split over the ranks, sub-batches sized by sharding.  Returns per-rank elapsed ms and the series count."""
    sptr = stream.cuda_stream
    mine = sharding.series_for_rank(n_series, rank, world)
    base = [workloads.config4_series(i).spectrum for i in range(32)]            # 32 distinct series (generation time) ...
    w0N = 1 << 22
    plan = fdas.Plan(w0N, ZMAX, DZ, SEGLEN, "bf16", stream=sptr)
    X = torch.from_numpy(np.stack([base[i % 32] for i in mine])).cuda()          # ... reused for series i, i+32, ...
    free_b, _ = torch.cuda.mem_get_info()
    sub = sharding.sub_batches(list(range(len(mine))), min(64, sharding.max_resident_series(plan.K, plan.M, 0, free_b)))
    cap = 1024
    peaks = torch.empty((len(mine), cap, 3), dtype=torch.int32, device="cuda")
    counts = torch.zeros(len(mine), dtype=torch.int32, device="cuda")

    def survey():
        for sb in sub:
            b0, nb = sb[0], len(sb)
            rc = fdas.fdas_search_batched(plan._h, X[b0].data_ptr(), 0, nb, THRESH, peaks[b0].data_ptr(), cap, counts[b0:].data_ptr(), sptr)
            assert rc == 0, rc

    with torch.cuda.stream(stream):
        survey()
        stream.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        survey()
        b.record(stream)
        stream.synchronize()
    ms = a.elapsed_time(b)
    found = int(counts.sum().item())
    K, M = plan.K, plan.M
    plan.close()
    return ms, len(mine), K, M, found, len(sub)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--noise-only", action="store_true", help="skip the (slow) signal injection; same shapes")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config block (configs 1, 2, 4, 5)")
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
    timer = Timer(torch, stream)
    results = {}
    peaks_dev = torch.empty(PEAK_CAPACITY * 3, dtype=torch.int32, device="cuda")
    count_dev = torch.zeros(1, dtype=torch.int32, device="cuda")
    x_dev = torch.from_numpy(w.spectrum).cuda()
    x_dev64 = None
    x_pin = torch.from_numpy(w.spectrum).pin_memory()
    peaks_pin = torch.empty(PEAK_CAPACITY * 3, dtype=torch.int32).pin_memory()
    sampler = None
    peak_gbs, peak_src, peaks_json = measured_peaks()
    tensor_peak = float(peaks_json.get("bf16_tflops", 1590.0))
    tensor_src = "measured (MEASURED_PEAKS.json bf16_tflops, burst)" if "bf16_tflops" in peaks_json else "fallback 1.59 PFLOP/s"
    sm_max = float(peaks_json.get("sm_max_mhz", 1965.0))
    alu_peak = 148 * 128 * 2 * sm_max * 1e6 / 1e12       # TFLOP/s fp32 FMA, DESIGN.md section 7

    # (name, precision, algorithm, plane format, plane-free step); headline (bf16, float plane) last so the clock sample covers it
    variants = (("f64", "f64", "fft", "f32", False), ("f32_fft", "f32", "fft", "f32", False), ("f32_split3", "f32", "auto", "f32", False),
                ("f32_split3_planefree", "f32", "auto", "f32", True), ("bf16_fft", "bf16", "fft", "f32", False),
                ("bf16_plane16", "bf16", "auto", "bf16", False), ("bf16_planefree", "bf16", "auto", "f32", True),
                ("bf16", "bf16", "auto", "f32", False))
    for name, pname, algo, pfmt, plane_free in variants:
        plan = fdas.Plan(w.N, ZMAX, DZ, SEGLEN, pname, stream=sptr, algorithm=algo, plane=pfmt)
        K, M, S, V = plan.K, plan.M, plan.S, int(plan.info.valid_per_seg)
        if pname == "f64" and x_dev64 is None:
            x_dev64 = x_dev.to(torch.complex128)
        xin = x_dev64 if pname == "f64" else x_dev
        plane = None if plane_free else torch.empty((K, M), dtype=plan.plane_dtype(), device="cuda")
        h = plan._h
        pptr = 0 if plane_free else plane.data_ptr()

        def step():
            rc = fdas.fdas_search(h, xin.data_ptr(), pptr, THRESH, peaks_dev.data_ptr(), PEAK_CAPACITY, count_dev.data_ptr(), sptr)
            assert rc == 0, rc

        def convolve_only():
            assert fdas.fdas_convolve(h, xin.data_ptr(), pptr, sptr) == 0

        reps = args.steps if name != "f64" else max(3, min(args.steps, 5))
        with torch.cuda.stream(stream):
            for _ in range(args.warmup if name != "f64" else 3):
                step()
            stream.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        if name == "bf16" and rank == 0:
            sampler = ClockSampler(local)
        l0 = plan.launch_count()
        step_ms = timer(step, reps)                 # the timed region: K steps of the whole hot path
        torch.cuda.synchronize()
        launches = plan.launch_count() - l0
        if world > 1:
            dist.barrier()
        # the dominant kernel alone (roofline): fdas_convolve, same stream, same flush
        conv_ms = step_ms if plane_free else timer(convolve_only, reps)
        info = plan.describe(plane, 1)
        extra = {}
        if pfmt == "bf16":                       # the paper's quick cast of the bf16-stored plane
            wide = torch.empty((K, M), dtype=torch.float32, device="cuda")
            extra["cast_ms"] = float(np.mean(timer(lambda: plan.quick_cast(plane, wide, stream=sptr), 5, warm=1)))
            del wide
        if name == "bf16":
            hs = torch.empty((K, M), dtype=torch.float32, device="cuda")   # NEXT-3: harmonic sums (4 harmonics) of the headline plane
            extra["hsum_ms"] = float(np.mean(timer(lambda: plan.harmonic_sum(plane, 4, hs, stream=sptr), 5, warm=1)))
            extra["hsum_drift_ms"] = float(np.mean(timer(lambda: plan.harmonic_sum(plane, 4, hs, stream=sptr, drift=True), 3, warm=1)))
            del hs
            ts = torch.randn(w.N, dtype=torch.float32, device="cuda")      # NEXT-4: the fp32 real FFT ahead of the convolution
            xo = torch.empty(M, dtype=torch.complex64, device="cuda")
            extra["rfft_ms"] = float(np.mean(timer(lambda: plan.spectrum(ts, xo, stream=sptr), 5, warm=1)))
            del ts, xo
            # a6 as a pass of its own (fdas_peaks over the stored plane) and the paper's harmonic-band maxima (Table 3)
            pk = torch.empty(3 * PEAK_CAPACITY, dtype=torch.int32, device="cuda")
            pc = torch.zeros(1, dtype=torch.int32, device="cuda")
            extra["peaks_ms"] = float(np.mean(timer(lambda: fdas.fdas_peaks(plan._h, plane.data_ptr(), THRESH, pk.data_ptr(), PEAK_CAPACITY,
                                                                             pc.data_ptr(), sptr), 5, warm=1)))
            bm = torch.empty(3 * 16, dtype=torch.int32, device="cuda")
            extra["band_ms"] = float(np.mean(timer(lambda: fdas.fdas_band_max(plan._h, plane.data_ptr(), BAND_F_BIN, 16, bm.data_ptr(), sptr),
                                                   5, warm=1)))
            del pk, pc, bm
            # NEXT-4: the jerk search as a volume: 5 slabs w = -8..8 of the same bank on the same spectrum,
            # every slab convolved and the 26-neighbour peak rule applied over (w, z, r), one library call
            with torch.cuda.stream(stream):
                vol = fdas.Volume(w.N, ZMAX, DZ, 8.0, 4.0, SEGLEN, "bf16", stream=sptr)
            vbuf = torch.empty((vol.W, vol.K, vol.M), dtype=torch.float32, device="cuda")
            vpk = torch.empty(4 * PEAK_CAPACITY, dtype=torch.int32, device="cuda")
            vct = torch.zeros(1, dtype=torch.int32, device="cuda")

            def vsearch():
                assert fdas.fdas_volume_search(vol._v, x_dev.data_ptr(), vbuf.data_ptr(), THRESH, vpk.data_ptr(), PEAK_CAPACITY,
                                               vct.data_ptr(), sptr) == 0

            extra["volume_ms"] = float(np.mean(timer(vsearch, 3, warm=1)))
            extra["volume_shape"] = [vol.W, vol.K, vol.M]
            extra["volume_peaks"] = int(vct.item())
            vol.close()
            del vbuf, vpk, vct
            torch.cuda.empty_cache()
        total_ms = sharding.max_over_ranks(float(sum(step_ms)), device="cuda")
        n_found = int(count_dev.item())
        res = dict(K=K, M=M, S=S, V=V, conv_ms=float(np.mean(conv_ms)), conv_ms_min=float(np.min(conv_ms)),
                   step_ms=total_ms / reps, launches=launches, steps=reps, n_found=n_found, info=info, **extra)

        # ---- end to end through the host-buffer entry points (H2D spectrum, search, D2H peak list)
        if name == "bf16":
            e2e_steps = max(3, min(args.steps, 10))
            for _ in range(2):
                n_e2e = plan.search_host(x_pin, THRESH, peaks_pin, PEAK_CAPACITY, sptr)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                n_e2e = plan.search_host(x_pin, THRESH, peaks_pin, PEAK_CAPACITY, sptr)
            torch.cuda.synchronize()
            res["e2e_s"] = sharding.max_over_ranks((time.perf_counter() - t0) / e2e_steps, device="cuda")
            res["n_e2e"] = n_e2e
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
            res["e2e_batched_s"] = sharding.max_over_ranks((time.perf_counter() - t0) / (3 * nb), device="cuda")
            del xb_pin, pk_pin, ct_pin
        results[name] = res
        del plane
        plan.close()
        torch.cuda.empty_cache()

    clocks = sampler.stop() if sampler else {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
    del x_dev64

    # ---- BASELINE.json config 4 as a plane-free survey (series split over the ranks by sharding.py)
    sv_ms, sv_n, sv_K, sv_M, sv_found, sv_sub = bench_config4_survey(fdas, workloads, sharding, torch, stream, rank, world)
    sv_ms = sharding.max_over_ranks(sv_ms, device="cuda")
    sv_total = int(sharding.sum_over_ranks(sv_n, device="cuda"))

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    configs = None
    if not args.no_configs:
        configs = bench_other_configs(fdas, workloads, torch, timer, sptr, peak_gbs, tensor_peak, alu_peak)
    configs = configs or {}
    configs["config4_survey_plane_free"] = {
        "note": "all 256 series of config 4 (32 distinct seeded series, each used 8 times) through the plane-free "
                "fdas_search_batched in sub-batches; no plane is written (256 planes would be 208 GB); series split over the ranks",
        "series": sv_total, "sub_batches_per_rank": sv_sub, "ms_total": sv_ms, "ms_per_series": sv_ms / max(1, sv_n),
        "points_per_s": sv_total * sv_K * sv_M / (sv_ms * 1e-3), "peaks_found_rank0": sv_found}

    r = results["bf16"]
    K, M, S, V = r["K"], r["M"], r["S"], r["V"]
    points = K * M
    value = world * points / (r["step_ms"] * 1e-3)
    alg_bytes = algorithmic_bytes(K, M, S, V)
    achieved = alg_bytes / (r["conv_ms"] * 1e-3) / 1e9
    flops = nominal_flops(K, M, S, V)

    def prec_entry(name, note, plane_elem=4, spec_elem=8):
        q = results[name]
        ab = algorithmic_bytes(K, M, S, V, plane_elem=plane_elem, spec_elem=spec_elem)
        e = {"kernel": q["info"]["kernel"], "algorithm": q["info"]["algorithm"], "grid": [q["info"]["grid_x"], q["info"]["grid_y"]],
             "work_item_bins": q["info"]["work_item_bins"], "convolve_ms": q["conv_ms"], "convolve_ms_min": q["conv_ms_min"],
             "step_ms": q["step_ms"], "steps": q["steps"], "points_per_s": points / (q["step_ms"] * 1e-3),
             "convolve_points_per_s": points / (q["conv_ms"] * 1e-3), "peaks_found": q["n_found"], "note": note}
        if plane_elem:
            e["hbm_gbs"] = ab / (q["conv_ms"] * 1e-3) / 1e9
            e["hbm_frac_of_measured_peak"] = e["hbm_gbs"] / peak_gbs
        if q["info"]["tensor_flops"] > 0:
            e["tensor_tflops_issued"] = q["info"]["tensor_flops"] / (q["conv_ms"] * 1e-3) / 1e12
            e["tensor_frac_of_measured_peak"] = e["tensor_tflops_issued"] / tensor_peak
        else:
            peak = alu_peak / 2 if name == "f64" else alu_peak
            e["alu_tflops_nominal"] = flops / (q["conv_ms"] * 1e-3) / 1e12
            e["alu_frac"] = e["alu_tflops_nominal"] / peak
        return e

    rp, rpf = results["bf16_plane16"], results["bf16_planefree"]
    precisions = {
        "bf16": prec_entry("bf16", "headline: bf16 spectrum and taps (RNE), fp32 accumulation on the tensor cores, float plane"),
        "bf16_planefree": prec_entry("bf16_planefree", "fdas_search with a NULL plane: scan launch + recheck launch, no plane in HBM (the whole step IS the "
                                     "kernel pair; convolve_ms = step_ms); bound by the tensor pipe", plane_elem=0),
        "bf16_plane16": prec_entry("bf16_plane16", "NEXT-1: bf16-stored plane (PAPER.md:91-93); fdas_quick_cast timed separately", plane_elem=2),
        "bf16_fft": prec_entry("bf16_fft", "FDAS_ALGO_FFT: the overlap-save FFT kernel with bf16 storage + separate peak pass"),
        "f32_split3": prec_entry("f32_split3", "FDAS_F32 default: NOT fp32 arithmetic -- every fp32 operand split into two bf16 terms, three products "
                                 "per tap on the tensor cores, fp32 accumulation (error ~3e-6 P_peak, tolerance 1e-4 P_peak)"),
        "f32_split3_planefree": prec_entry("f32_split3_planefree", "plane-free search of the split-operand form", plane_elem=0),
        "f32_fft": prec_entry("f32_fft", "true fp32 arithmetic: the overlap-save FFT kernel (PAPER.md:65-67) + separate peak pass"),
        "f64": prec_entry("f64", "the paper's gold standard (PAPER.md:15, :315): fp64 overlap-save FFT kernel, double plane + separate peak pass",
                          plane_elem=8, spec_elem=16),
    }
    precisions["bf16_plane16"]["quick_cast_ms"] = rp["cast_ms"]
    precisions["bf16_plane16"]["quick_cast_hbm_gbs"] = 6.0 * points / (rp["cast_ms"] * 1e-3) / 1e9
    precisions["bf16_plane16"]["convolve_plus_quick_cast_ms"] = rp["conv_ms"] + rp["cast_ms"]
    speedups = {
        "bf16_over_f32_split3": results["f32_split3"]["conv_ms"] / r["conv_ms"],
        "bf16_over_f32_fft": results["f32_fft"]["conv_ms"] / r["conv_ms"],
        "bf16_fft_over_f32_fft": results["f32_fft"]["conv_ms"] / results["bf16_fft"]["conv_ms"],
        "bf16_over_f64": results["f64"]["conv_ms"] / r["conv_ms"],
        "bf16_planefree_over_bf16_whole_step": r["step_ms"] / rpf["step_ms"],
        "paper_bf16_over_fp32": "~1.6x on 'NVIDIA Ampere' (PAPER.md:15; context, not the target)",
    }
    others = {
        "harmonic_sum_4": {"ms": r["hsum_ms"], "algorithmic_gbs": hsum_bytes(K, M, 4) / (r["hsum_ms"] * 1e-3) / 1e9,
                           "note": "NEXT-3: fdas_harmonic_sum, 4 harmonics, on the headline float plane; bytes = elements read + plane written"},
        "harmonic_sum_drift_4": {"ms": r["hsum_drift_ms"], "note": "fdas_harmonic_sum_drift, 4 harmonics (window maxima, reading A26)"},
        "peaks_pass": {"ms": r["peaks_ms"], "algorithmic_gbs": 4.0 * K * M / (r["peaks_ms"] * 1e-3) / 1e9,
                       "note": "a6 as its own pass: fdas_peaks over the stored float plane (one read of the plane)"},
        "band_max_16": {"ms": r["band_ms"], "algorithmic_gbs": 4.0 * K * min(M, int(16.5 * BAND_F_BIN) + 1) / (r["band_ms"] * 1e-3) / 1e9,
                        "note": "fdas_band_max (PAPER.md Table 3): maxima of 16 harmonic bands of a %g-bin fundamental; bytes = the band columns read" % BAND_F_BIN},
        "real_fft": {"ms": r["rfft_ms"], "algorithmic_gbs": 6.0 * 4 * M / (r["rfft_ms"] * 1e-3) / 1e9,
                     "note": "NEXT-4: fdas_spectrum, fp32 real FFT of the 2^23-sample series (outside the timed step, as in the paper); "
                             "bytes = series read + spectrum written"},
        "jerk_volume_search": {"ms": r["volume_ms"], "shape_w_k_m": r["volume_shape"], "peaks_found": r["volume_peaks"],
                               "points_per_s": float(np.prod(r["volume_shape"])) / (r["volume_ms"] * 1e-3),
                               "note": "NEXT-4: fdas_volume_search, bf16: 5 jerk slabs (w = -8..8 step 4) x 97 templates x 2^22 bins, float volume "
                                       "written + 26-neighbour peak rule over (w, z, r)"},
    }

    cpu = None
    if not args.no_cpu_baseline:
        v, dt, cores, desc = time_oracle_sample(w.spectrum, 1 << 22)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}

    kern = r["info"]["kernel"]
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
                "api": "fdas_search_host (pinned host spectrum in, peak list out; plane-free on the device)", "ms_per_step": r["e2e_s"] * 1e3,
                "batched": {"value": world * points / r["e2e_batched_s"], "unit": UNIT, "ms_per_series": r["e2e_batched_s"] * 1e3,
                            "series_per_call": 8, "h2d_bytes_per_series": int(M * 8), "d2h_bytes_per_series": 4 + 12 * 4096,
                            "api": "fdas_search_host_batched (8 pinned host spectra per call; copy of series i+1 overlaps the search of series i)"}},
        "gpu_launches": int(r["launches"]),
        "roofline": {"bound": "hbm", "kernel": kern + " (fdas_convolve, bf16; name and grid from fdas_describe_convolve)", "achieved": achieved,
                     "peak": peak_gbs, "unit": "GB/s", "frac": achieved / peak_gbs, "traffic": dram_traffic_of(kern),
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
                     "kernel_ms": r["conv_ms"], "kernel_ms_min": r["conv_ms_min"], "frac_of_nominal_8TBs": achieved / 8000.0,
                     "grid": [r["info"]["grid_x"], r["info"]["grid_y"]], "block_threads": r["info"]["block_threads"],
                     "tensor_tflops_issued": r["info"]["tensor_flops"] / (r["conv_ms"] * 1e-3) / 1e12,
                     "tensor_frac_of_measured_peak": r["info"]["tensor_flops"] / (r["conv_ms"] * 1e-3) / 1e12 / tensor_peak,
                     "per_precision": precisions, "per_config": configs},
        "roofline_planefree": {"bound": "tensor", "kernel": rpf["info"]["kernel"], "achieved": rpf["info"]["tensor_flops"] / (rpf["step_ms"] * 1e-3) / 1e12,
                               "peak": tensor_peak, "unit": "TFLOP/s", "frac": rpf["info"]["tensor_flops"] / (rpf["step_ms"] * 1e-3) / 1e12 / tensor_peak,
                               "flops_per_launch": rpf["info"]["tensor_flops"], "peak_source": tensor_src, "step_ms": rpf["step_ms"],
                               "count": "issued dense MMA flops of the scan launch (tiles x 2 parts x K steps x 2*128*N*16, padding included), "
                                        "over the time of BOTH launches (scan + recheck)"},
        "cpu_baseline": cpu,
        "precisions": precisions,
        "speedups": speedups,
        "other_kernels": others,
        "configs": configs,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
