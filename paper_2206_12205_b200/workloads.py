"""Seeded synthetic workloads (BASELINE.json configs 1-5; recipe in DESIGN.md section 4).

numpy only.  This module holds NONE of the method's arithmetic (no template, no
convolution, no overlap-save): it draws a noisy time series, injects constant-fdot tones
in the TIME domain, and takes the fp32 real FFT that the paper keeps outside the
accelerated section ("The 'Real FFT' ... was intentionally left in single-precision",
PAPER.md:85).  The oracle and the CUDA path both consume the complex64 spectrum it returns.

The paper's own inputs (SIGPROC ``fake`` filterbanks; GMRT data, :301) are
not available; these seeded series stand in for them.

Conventions (readings A2, A3, A8, A9):
* z > 0  <=> frequency increasing with time; r0 is the MEAN (mid-observation) frequency in
  Fourier bins; phase phi(u) = 2 pi [(r0 - z/2) u + (z/2) u^2] + phi0, u = n/N.
* a tone of amplitude a has coherent power |A|^2 = a^2 N / 4 in unit-noise units, so
  power p  <=>  a = 2 sqrt(p/N).
* spectrum = rfft(x) / sqrt(N), bins 0..N/2-1 (Nyquist dropped), complex64; the noise has
  sigma = 1 so the mean noise power per bin is 1 (analytic scale, not an estimate).
* draw order from ``numpy.random.default_rng(seed)``: noise first, then per signal
  (r0 or f_spin, z, power, phi0).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Iterator, List, Optional

import numpy as np

TSAMP_CONFIG3 = 64e-6  # s (BASELINE.json config 3: "about 537 s at 64 us sampling")


@dataclasses.dataclass
class Injection:
    r0: float        # mean frequency, Fourier bins
    z: float         # drift over the observation, Fourier bins
    power: float     # coherent power |A|^2 in unit-noise units (fundamental)
    phi0: float      # radians
    harmonic: int = 1


@dataclasses.dataclass
class Workload:
    name: str
    N: int                 # real samples per series
    zmax: float
    dz: float
    seglen: int
    spectrum: np.ndarray   # complex64 [M] (or [B, M] for a batch)
    injections: List[Injection]
    seed: int
    series: Optional[np.ndarray] = None   # the fp32 time series itself, kept on request (inputs of fdas_spectrum)

    @property
    def M(self) -> int:
        return self.N // 2

    @property
    def K(self) -> int:
        return 2 * int(math.floor(self.zmax / self.dz + 1e-9)) + 1


def _add_tone(x: np.ndarray, r0: float, z: float, power: float, phi0: float,
              harmonics=None, chunk: int = 1 << 20, w: float = 0.0) -> None:
    """x += sum_h a_h cos(h * theta(u)), theta(u) = 2 pi[(r0 - z/2)u + (z/2)u^2] + phi0.

    ``harmonics`` = list of (h, relative amplitude); default a single fundamental.  The
    phase is evaluated in fp64 (reduced modulo 1 cycle before the cosine) and the sum is
    added into the fp32 series.  Harmonic h of the train sits at (h r0, h z).
    """
    N = len(x)
    a1 = 2.0 * math.sqrt(power / N)
    if harmonics is None:
        harmonics = [(1, 1.0)]
    for s in range(0, N, chunk):
        e = min(N, s + chunk)
        u = np.arange(s, e, dtype=np.float64) / N
        cyc = (r0 - 0.5 * z) * u + 0.5 * z * u * u + phi0 / (2.0 * math.pi)
        if w != 0.0:   # jerk: frequency r0 + z (u - 1/2) + (w/2)(u^2 - u + 1/6); phase term (w/12)(2u^3 - 3u^2 + u)
            cyc += (w / 12.0) * (2.0 * u * u * u - 3.0 * u * u + u)
        cyc -= np.floor(cyc)
        acc = np.zeros(e - s, dtype=np.float64)
        for h, rel in harmonics:
            acc += (a1 * rel) * np.cos((2.0 * math.pi * h) * cyc)
        x[s:e] += acc.astype(np.float32)


def spectrum_of(x: np.ndarray) -> np.ndarray:
    """fp32 real FFT, bins 0..N/2-1, scaled 1/sqrt(N) (unit mean noise power), complex64."""
    N = len(x)
    X = np.fft.rfft(x.astype(np.float32, copy=False))
    X = X[: N // 2] * (1.0 / math.sqrt(N))
    return np.ascontiguousarray(X.astype(np.complex64))


def _noise(rng: np.random.Generator, N: int) -> np.ndarray:
    return rng.standard_normal(N, dtype=np.float32)


def config1(noise: bool = True, keep_series: bool = False) -> Workload:
    """Tiny series: N=2^16, seed 1, one tone r0=10000.25, z=+20, power 100; K=21, S=1024.

    ``noise=False`` gives the noise-free twin used by the closed-form pin (reading A19).
    """
    N, seed = 1 << 16, 1
    rng = np.random.default_rng(seed)
    x = _noise(rng, N)
    if not noise:
        x = np.zeros(N, dtype=np.float32)
    inj = Injection(r0=10000.25, z=20.0, power=100.0, phi0=0.0)
    _add_tone(x, inj.r0, inj.z, inj.power, inj.phi0)
    return Workload("config1", N, 20.0, 2.0, 1024, spectrum_of(x), [inj], seed, series=x if keep_series else None)


def _draw_tones(rng, n, r_lo, r_hi, z_lo, z_hi) -> List[Injection]:
    out = []
    for _ in range(n):
        r0 = rng.uniform(r_lo, r_hi)
        z = rng.uniform(z_lo, z_hi)
        p = math.exp(rng.uniform(math.log(30.0), math.log(300.0)))
        phi0 = rng.uniform(0.0, 2.0 * math.pi)
        out.append(Injection(float(r0), float(z), float(p), float(phi0)))
    return out


def config2() -> Workload:
    """N=2^20, seed 2, 8 tones r0~U[1000,5e5], z~U[-90,90], power logU[30,300]; K=97, S=2048."""
    N, seed = 1 << 20, 2
    rng = np.random.default_rng(seed)
    x = _noise(rng, N)
    inj = _draw_tones(rng, 8, 1000.0, 5e5, -90.0, 90.0)
    for t in inj:
        _add_tone(x, t.r0, t.z, t.power, t.phi0)
    return Workload("config2", N, 96.0, 2.0, 2048, spectrum_of(x), inj, seed)


def config3(n_trains: int = 64) -> Workload:
    """N=2^23, seed 3, 64 pulse trains with a 5-harmonic Gaussian profile (5 % FWHM duty
    cycle), f_spin~U[10,500] Hz at 64 us sampling, z~U[-96,96]; K=97, S=2048.

    Harmonic amplitudes a_h = a_1 exp(-2 pi^2 sigma^2 (h^2-1)), sigma = 0.05/(2 sqrt(2 ln 2))
    (Fourier series of a Gaussian pulse).  Fundamental power logU[30,300] (reading A20).
    """
    N, seed = 1 << 23, 3
    T = N * TSAMP_CONFIG3
    rng = np.random.default_rng(seed)
    x = _noise(rng, N)
    sigma = 0.05 / (2.0 * math.sqrt(2.0 * math.log(2.0)))
    harm = [(h, math.exp(-2.0 * math.pi ** 2 * sigma ** 2 * (h * h - 1))) for h in range(1, 6)]
    inj: List[Injection] = []
    for _ in range(n_trains):
        f = rng.uniform(10.0, 500.0)
        z = rng.uniform(-96.0, 96.0)
        p = math.exp(rng.uniform(math.log(30.0), math.log(300.0)))
        phi0 = rng.uniform(0.0, 2.0 * math.pi)
        r0 = f * T
        _add_tone(x, r0, z, p, phi0, harmonics=harm)
        for h, rel in harm:
            inj.append(Injection(float(h * r0), float(h * z), float(p * rel * rel),
                                 float(h * phi0), harmonic=h))
    return Workload("config3", N, 96.0, 2.0, 2048, spectrum_of(x), inj, seed)


def config4_series(i: int) -> Workload:
    """Series i (0..255) of the batched config: N=2^22, seed 100+i; series with i % 10 == 0
    carry one tone drawn as in config 2 (reading A20).  K=97, S=2048."""
    N, seed = 1 << 22, 100 + i
    rng = np.random.default_rng(seed)
    x = _noise(rng, N)
    inj: List[Injection] = []
    if i % 10 == 0:
        inj = _draw_tones(rng, 1, 1000.0, 5e5, -90.0, 90.0)
        for t in inj:
            _add_tone(x, t.r0, t.z, t.power, t.phi0)
    return Workload(f"config4[{i}]", N, 96.0, 2.0, 2048, spectrum_of(x), inj, seed)


def config4(indices=range(256)) -> Iterator[Workload]:
    for i in indices:
        yield config4_series(i)


def config5() -> Workload:
    """N=2^23, seed 4, 32 tones z~U[-190,190], r0~U[1e4, M-1e4], power logU[30,300];
    K=201 (z in [-200,200] step 2), S=4096."""
    N, seed = 1 << 23, 4
    M = N // 2
    rng = np.random.default_rng(seed)
    x = _noise(rng, N)
    inj = _draw_tones(rng, 32, 1e4, M - 1e4, -190.0, 190.0)
    for t in inj:
        _add_tone(x, t.r0, t.z, t.power, t.phi0)
    return Workload("config5", N, 200.0, 2.0, 4096, spectrum_of(x), inj, seed)


def harmonic_train(N: int, seed: int, r0: float, z: float, power: float, rel_amplitudes, zmax: float = 20.0,
                   dz: float = 2.0, seglen: int = 1024, noise: bool = True) -> Workload:
    """One pulse train whose harmonic h = 1.. has amplitude rel_amplitudes[h-1] (relative to the
    fundamental of coherent power ``power``) and sits at (h r0, h z): input of the harmonic-sum tests."""
    rng = np.random.default_rng(seed)
    x = _noise(rng, N) if noise else np.zeros(N, dtype=np.float32)
    inj = Injection(float(r0), float(z), float(power), 0.0)
    _add_tone(x, r0, z, power, 0.0, harmonics=[(h + 1, float(a)) for h, a in enumerate(rel_amplitudes)])
    return Workload("harmonic_train", N, zmax, dz, seglen, spectrum_of(x), [inj], seed)


def jerk_tone(N: int, seed: int, r0: float, z: float, w: float, power: float, zmax: float = 20.0, dz: float = 2.0,
              seglen: int = 1024, noise: bool = True) -> Workload:
    """One tone with drift z and jerk w (both in Fourier bins over the observation), mean frequency r0."""
    rng = np.random.default_rng(seed)
    x = _noise(rng, N) if noise else np.zeros(N, dtype=np.float32)
    _add_tone(x, r0, z, power, 0.0, w=w)
    return Workload("jerk_tone", N, zmax, dz, seglen, spectrum_of(x), [Injection(float(r0), float(z), float(power), 0.0)], seed)


def noise_only(N: int, seed: int, zmax: float = 96.0, dz: float = 2.0, seglen: int = 2048) -> Workload:
    """White-noise series of any length (throughput runs and the chi^2_2 invariant)."""
    rng = np.random.default_rng(seed)
    return Workload(f"noise(N={N},seed={seed})", N, zmax, dz, seglen,
                    spectrum_of(_noise(rng, N)), [], seed)


def by_name(name: str) -> Workload:
    return {"config1": config1, "config2": config2, "config3": config3, "config5": config5}[name]()
