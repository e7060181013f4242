"""Thin ctypes binding over libfdas (include/fdas.h).  Argument marshalling only: every step
of the path runs in the CUDA library.  The functions carry the C names; ``Plan`` is a small
convenience wrapper that owns a plan handle and passes torch tensors' ``data_ptr()``.

There is no CPU fallback: if ``libfdas.so`` has not been built, importing the library raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdas.so")

FDAS_F64, FDAS_F32, FDAS_BF16 = 0, 1, 2
FDAS_OK, FDAS_ERR_INVALID_ARG, FDAS_ERR_ALLOC, FDAS_ERR_CUDA, FDAS_ERR_NOT_BUILT, FDAS_ERR_UNSUPPORTED, FDAS_ERR_TOO_LARGE = range(7)
FDAS_SEARCH_STATIC_MAX_BINS = 1 << 22
PRECISIONS = {"f64": FDAS_F64, "f32": FDAS_F32, "bf16": FDAS_BF16}
FDAS_ALGO_AUTO, FDAS_ALGO_FFT, FDAS_ALGO_MMA, FDAS_ALGO_MMA_SCALAR = 0, 1, 2, 3
ALGORITHMS = {"auto": FDAS_ALGO_AUTO, "fft": FDAS_ALGO_FFT, "mma": FDAS_ALGO_MMA,
              "mma_scalar": FDAS_ALGO_MMA_SCALAR}
FDAS_PLANE_F32, FDAS_PLANE_BF16 = 0, 1
PLANE_FORMATS = {"f32": FDAS_PLANE_F32, "bf16": FDAS_PLANE_BF16}

EXPORTS = [
    "fdas_plan_create", "fdas_plan_destroy", "fdas_plan_info", "fdas_z_of_index",
    "fdas_build_templates", "fdas_convolve", "fdas_convolve_batched", "fdas_peaks",
    "fdas_convolve_host", "fdas_search_host", "fdas_templates_host", "fdas_taps_host",
    "fdas_launch_count", "fdas_status_string", "fdas_last_cuda_error",
    "fdas_set_algorithm", "fdas_get_algorithm", "fdas_tapmatrix_host", "fdas_search",
    "fdas_set_plane_format", "fdas_get_plane_format", "fdas_quick_cast", "fdas_harmonic_sum", "fdas_harmonic_sum_drift", "fdas_band_max", "fdas_search_host_batched", "fdas_spectrum", "fdas_plan_create_jerk",
    "fdas_search_batched", "fdas_describe_convolve", "fdas_search_host_timeseries", "fdas_search_host_timeseries_batched",
    "fdas_volume_create", "fdas_volume_destroy", "fdas_volume_info", "fdas_volume_w_of_index", "fdas_volume_slab",
    "fdas_volume_set_algorithm", "fdas_volume_build_templates", "fdas_volume_convolve", "fdas_volume_peaks",
    "fdas_volume_search", "fdas_volume_search_host", "fdas_volume_launch_count", "fdas_volume_last_cuda_error",
    "fdas_search_static",
]


class fdas_peak_t(ctypes.Structure):
    _fields_ = [("z_index", ctypes.c_int32), ("r", ctypes.c_int32), ("power", ctypes.c_float)]


class fdas_info_t(ctypes.Structure):
    _fields_ = [
        ("n_bins", ctypes.c_int64), ("n_templates", ctypes.c_int32), ("seglen", ctypes.c_int32),
        ("halfwidth_max", ctypes.c_int32), ("overlap_left", ctypes.c_int32),
        ("valid_per_seg", ctypes.c_int32), ("precision", ctypes.c_int32),
        ("n_segments", ctypes.c_int64), ("plane_row_pitch", ctypes.c_int64),
        ("plane_elem_bytes", ctypes.c_size_t), ("spectrum_elem_bytes", ctypes.c_size_t),
        ("bank_bytes", ctypes.c_size_t),
    ]


class fdas_peak3_t(ctypes.Structure):
    _fields_ = [("w_index", ctypes.c_int32), ("z_index", ctypes.c_int32), ("r", ctypes.c_int32), ("power", ctypes.c_float)]


class fdas_volume_info_t(ctypes.Structure):
    _fields_ = [("n_slabs", ctypes.c_int32), ("n_templates", ctypes.c_int32), ("n_bins", ctypes.c_int64),
                ("precision", ctypes.c_int32), ("elem_bytes", ctypes.c_size_t), ("wmax", ctypes.c_double), ("dw", ctypes.c_double)]


class fdas_kernel_info_t(ctypes.Structure):
    _fields_ = [
        ("algorithm", ctypes.c_int32), ("split", ctypes.c_int32), ("groups", ctypes.c_int32), ("nch", ctypes.c_int32),
        ("k_steps", ctypes.c_int32), ("work_item_bins", ctypes.c_int32), ("grid_x", ctypes.c_int32),
        ("grid_y", ctypes.c_int32), ("block_threads", ctypes.c_int32), ("dynamic_smem_bytes", ctypes.c_size_t),
        ("tensor_flops", ctypes.c_double), ("kernel", ctypes.c_char * 128),
    ]


_lib: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Loads libfdas.so; raises if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} not found: build it with `python -m paper_2206_12205_b200._build` "
            "(or __graft_entry__.build()); libfdas has no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i, i64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_double
    L.fdas_plan_create.argtypes = [ctypes.POINTER(vp), i64, dbl, dbl, i, i]
    L.fdas_plan_create_jerk.argtypes = [ctypes.POINTER(vp), i64, dbl, dbl, dbl, i, i]
    L.fdas_plan_destroy.argtypes = [vp]
    L.fdas_plan_info.argtypes = [vp, ctypes.POINTER(fdas_info_t)]
    L.fdas_z_of_index.argtypes = [vp, i, ctypes.POINTER(dbl)]
    L.fdas_build_templates.argtypes = [vp, vp]
    L.fdas_convolve.argtypes = [vp, vp, vp, vp]
    L.fdas_convolve_batched.argtypes = [vp, vp, vp, i, vp]
    L.fdas_peaks.argtypes = [vp, vp, ctypes.c_float, vp, i, vp, vp]
    L.fdas_search.argtypes = [vp, vp, vp, ctypes.c_float, vp, i, vp, vp]
    L.fdas_search_batched.argtypes = [vp, vp, vp, i, ctypes.c_float, vp, i, vp, vp]
    L.fdas_search_static.argtypes = [vp, vp, ctypes.c_float, vp, i, vp, vp]
    L.fdas_volume_create.argtypes = [ctypes.POINTER(vp), i64, dbl, dbl, dbl, dbl, i, i]
    L.fdas_volume_destroy.argtypes = [vp]
    L.fdas_volume_info.argtypes = [vp, ctypes.POINTER(fdas_volume_info_t)]
    L.fdas_volume_w_of_index.argtypes = [vp, i, ctypes.POINTER(dbl)]
    L.fdas_volume_slab.argtypes = [vp, i, ctypes.POINTER(vp)]
    L.fdas_volume_set_algorithm.argtypes = [vp, i]
    L.fdas_volume_build_templates.argtypes = [vp, vp]
    L.fdas_volume_convolve.argtypes = [vp, vp, vp, vp]
    L.fdas_volume_peaks.argtypes = [vp, vp, ctypes.c_float, vp, i, vp, vp]
    L.fdas_volume_search.argtypes = [vp, vp, vp, ctypes.c_float, vp, i, vp, vp]
    L.fdas_volume_search_host.argtypes = [vp, vp, ctypes.c_float, vp, i, ctypes.POINTER(i), vp]
    L.fdas_volume_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
    L.fdas_volume_last_cuda_error.argtypes = [vp]
    L.fdas_describe_convolve.argtypes = [vp, vp, i, ctypes.POINTER(fdas_kernel_info_t)]
    L.fdas_convolve_host.argtypes = [vp, vp, vp, vp]
    L.fdas_search_host.argtypes = [vp, vp, ctypes.c_float, vp, i, ctypes.POINTER(i), vp]
    L.fdas_templates_host.argtypes = [vp, vp, ctypes.c_size_t]
    L.fdas_taps_host.argtypes = [vp, vp, ctypes.c_size_t]
    L.fdas_tapmatrix_host.argtypes = [vp, vp, ctypes.c_size_t]
    L.fdas_set_algorithm.argtypes = [vp, i]
    L.fdas_get_algorithm.argtypes = [vp, ctypes.POINTER(i)]
    L.fdas_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
    L.fdas_set_plane_format.argtypes = [vp, i]
    L.fdas_get_plane_format.argtypes = [vp, ctypes.POINTER(i)]
    L.fdas_quick_cast.argtypes = [vp, vp, vp, i, vp]
    L.fdas_harmonic_sum.argtypes = [vp, vp, vp, i, vp]
    L.fdas_harmonic_sum_drift.argtypes = [vp, vp, vp, i, vp]
    L.fdas_band_max.argtypes = [vp, vp, dbl, i, vp, vp]
    L.fdas_spectrum.argtypes = [vp, vp, vp, vp]
    L.fdas_search_host_batched.argtypes = [vp, vp, i, ctypes.c_float, vp, i, vp, vp]
    L.fdas_search_host_timeseries.argtypes = [vp, vp, ctypes.c_float, vp, i, ctypes.POINTER(i), vp]
    L.fdas_search_host_timeseries_batched.argtypes = [vp, vp, i, ctypes.c_float, vp, i, vp, vp]
    L.fdas_status_string.argtypes = [i]
    L.fdas_status_string.restype = ctypes.c_char_p
    L.fdas_last_cuda_error.argtypes = [vp]
    for name in EXPORTS:
        if name != "fdas_status_string":
            getattr(L, name).restype = i
    _lib = L
    return L


class FdasError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_error: int = 0):
        self.status = status
        self.cuda_error = cuda_error
        msg = lib().fdas_status_string(status).decode()
        super().__init__(f"{where}: {msg}" + (f" (cudaError {cuda_error})" if cuda_error else ""))


# ---- the C entry points under their own names (raw: return the status code) -------------
def fdas_plan_create(N, zmax, dz, seglen, precision):
    h = ctypes.c_void_p()
    rc = lib().fdas_plan_create(ctypes.byref(h), int(N), float(zmax), float(dz), int(seglen), int(precision))
    return rc, h


def fdas_plan_create_jerk(N, zmax, dz, w, seglen, precision):
    h = ctypes.c_void_p()
    rc = lib().fdas_plan_create_jerk(ctypes.byref(h), int(N), float(zmax), float(dz), float(w), int(seglen), int(precision))
    return rc, h


def fdas_plan_destroy(h):
    return lib().fdas_plan_destroy(h)


def fdas_plan_info(h):
    info = fdas_info_t()
    rc = lib().fdas_plan_info(h, ctypes.byref(info))
    return rc, info


def fdas_z_of_index(h, k):
    z = ctypes.c_double()
    rc = lib().fdas_z_of_index(h, int(k), ctypes.byref(z))
    return rc, z.value


def fdas_build_templates(h, stream=0):
    return lib().fdas_build_templates(h, ctypes.c_void_p(stream))


def fdas_convolve(h, spectrum_ptr, plane_ptr, stream=0):
    return lib().fdas_convolve(h, ctypes.c_void_p(spectrum_ptr), ctypes.c_void_p(plane_ptr), ctypes.c_void_p(stream))


def fdas_convolve_batched(h, spectra_ptr, planes_ptr, batch, stream=0):
    return lib().fdas_convolve_batched(h, ctypes.c_void_p(spectra_ptr), ctypes.c_void_p(planes_ptr), int(batch),
                                       ctypes.c_void_p(stream))


def fdas_peaks(h, plane_ptr, threshold, peaks_ptr, capacity, count_ptr, stream=0):
    return lib().fdas_peaks(h, ctypes.c_void_p(plane_ptr), float(threshold), ctypes.c_void_p(peaks_ptr),
                            int(capacity), ctypes.c_void_p(count_ptr), ctypes.c_void_p(stream))


def fdas_search(h, spectrum_ptr, plane_ptr, threshold, peaks_ptr, capacity, count_ptr, stream=0):
    return lib().fdas_search(h, ctypes.c_void_p(spectrum_ptr), ctypes.c_void_p(plane_ptr), float(threshold),
                             ctypes.c_void_p(peaks_ptr), int(capacity), ctypes.c_void_p(count_ptr),
                             ctypes.c_void_p(stream))


def fdas_search_static(h, spectrum_ptr, threshold, peaks_ptr, capacity, count_ptr, stream=0):
    return lib().fdas_search_static(h, ctypes.c_void_p(spectrum_ptr), float(threshold), ctypes.c_void_p(peaks_ptr),
                                    int(capacity), ctypes.c_void_p(count_ptr), ctypes.c_void_p(stream))


def fdas_search_batched(h, spectra_ptr, planes_ptr, batch, threshold, peaks_ptr, capacity, counts_ptr, stream=0):
    return lib().fdas_search_batched(h, ctypes.c_void_p(spectra_ptr), ctypes.c_void_p(planes_ptr), int(batch), float(threshold),
                                     ctypes.c_void_p(peaks_ptr), int(capacity), ctypes.c_void_p(counts_ptr),
                                     ctypes.c_void_p(stream))


def fdas_convolve_host(h, spectrum_host_ptr, plane_host_ptr, stream=0):
    return lib().fdas_convolve_host(h, ctypes.c_void_p(spectrum_host_ptr), ctypes.c_void_p(plane_host_ptr),
                                    ctypes.c_void_p(stream))


def fdas_search_host(h, spectrum_host_ptr, threshold, peaks_host_ptr, capacity, stream=0):
    n = ctypes.c_int(0)
    rc = lib().fdas_search_host(h, ctypes.c_void_p(spectrum_host_ptr), float(threshold),
                                ctypes.c_void_p(peaks_host_ptr), int(capacity), ctypes.byref(n),
                                ctypes.c_void_p(stream))
    return rc, n.value


def fdas_templates_host(h, dst_ptr, nbytes):
    return lib().fdas_templates_host(h, ctypes.c_void_p(dst_ptr), int(nbytes))


def fdas_taps_host(h, dst_ptr, nbytes):
    return lib().fdas_taps_host(h, ctypes.c_void_p(dst_ptr), int(nbytes))


def fdas_tapmatrix_host(h, dst_ptr, nbytes):
    return lib().fdas_tapmatrix_host(h, ctypes.c_void_p(dst_ptr), int(nbytes))


def fdas_set_algorithm(h, algorithm):
    return lib().fdas_set_algorithm(h, int(algorithm))


def fdas_get_algorithm(h):
    a = ctypes.c_int(-1)
    rc = lib().fdas_get_algorithm(h, ctypes.byref(a))
    return rc, a.value


def fdas_set_plane_format(h, fmt):
    return lib().fdas_set_plane_format(h, int(fmt))


def fdas_get_plane_format(h):
    out = ctypes.c_int(0)
    rc = lib().fdas_get_plane_format(h, ctypes.byref(out))
    return rc, out.value


def fdas_quick_cast(h, plane_bf16_ptr, plane_f32_ptr, batch=1, stream=0):
    return lib().fdas_quick_cast(h, plane_bf16_ptr, plane_f32_ptr, int(batch), stream)


def fdas_harmonic_sum(h, plane_ptr, sum_ptr, n_harmonics, stream=0):
    return lib().fdas_harmonic_sum(h, plane_ptr, sum_ptr, int(n_harmonics), stream)


def fdas_harmonic_sum_drift(h, plane_ptr, sum_ptr, n_harmonics, stream=0):
    return lib().fdas_harmonic_sum_drift(h, plane_ptr, sum_ptr, int(n_harmonics), stream)


def fdas_band_max(h, plane_ptr, f_bin, n_bands, out_ptr, stream=0):
    return lib().fdas_band_max(h, plane_ptr, float(f_bin), int(n_bands), out_ptr, stream)


def fdas_search_host_batched(h, spectra_host_ptr, n_series, threshold, peaks_host_ptr, capacity, counts_host_ptr, stream=0):
    return lib().fdas_search_host_batched(h, spectra_host_ptr, int(n_series), threshold, peaks_host_ptr, int(capacity),
                                          counts_host_ptr, stream)


def fdas_search_host_timeseries(h, timeseries_host_ptr, threshold, peaks_host_ptr, capacity, stream=0):
    n = ctypes.c_int(0)
    rc = lib().fdas_search_host_timeseries(h, ctypes.c_void_p(timeseries_host_ptr), float(threshold),
                                           ctypes.c_void_p(peaks_host_ptr), int(capacity), ctypes.byref(n), ctypes.c_void_p(stream))
    return rc, n.value


def fdas_search_host_timeseries_batched(h, timeseries_host_ptr, n_series, threshold, peaks_host_ptr, capacity, counts_host_ptr, stream=0):
    return lib().fdas_search_host_timeseries_batched(h, timeseries_host_ptr, int(n_series), threshold, peaks_host_ptr, int(capacity),
                                                     counts_host_ptr, stream)


def fdas_spectrum(h, timeseries_ptr, spectrum_ptr, stream=0):
    return lib().fdas_spectrum(h, timeseries_ptr, spectrum_ptr, stream)


def fdas_describe_convolve(h, plane_ptr, batch=1):
    info = fdas_kernel_info_t()
    rc = lib().fdas_describe_convolve(h, ctypes.c_void_p(plane_ptr), int(batch), ctypes.byref(info))
    return rc, info


def fdas_launch_count(h):
    n = ctypes.c_int64()
    rc = lib().fdas_launch_count(h, ctypes.byref(n))
    return rc, n.value


def fdas_status_string(status):
    return lib().fdas_status_string(int(status)).decode()


def fdas_last_cuda_error(h):
    return lib().fdas_last_cuda_error(h)


# ---- f-fdot-fddot volume (jerk search) ----------------------------------------------------
def fdas_volume_create(N, zmax, dz, wmax, dw, seglen, precision):
    h = ctypes.c_void_p()
    rc = lib().fdas_volume_create(ctypes.byref(h), int(N), float(zmax), float(dz), float(wmax), float(dw), int(seglen), int(precision))
    return rc, h


def fdas_volume_destroy(v):
    return lib().fdas_volume_destroy(v)


def fdas_volume_info(v):
    info = fdas_volume_info_t()
    rc = lib().fdas_volume_info(v, ctypes.byref(info))
    return rc, info


def fdas_volume_w_of_index(v, i):
    w = ctypes.c_double()
    rc = lib().fdas_volume_w_of_index(v, int(i), ctypes.byref(w))
    return rc, w.value


def fdas_volume_slab(v, i):
    h = ctypes.c_void_p()
    rc = lib().fdas_volume_slab(v, int(i), ctypes.byref(h))
    return rc, h


def fdas_volume_set_algorithm(v, algorithm):
    return lib().fdas_volume_set_algorithm(v, int(algorithm))


def fdas_volume_build_templates(v, stream=0):
    return lib().fdas_volume_build_templates(v, ctypes.c_void_p(stream))


def fdas_volume_convolve(v, spectrum_ptr, volume_ptr, stream=0):
    return lib().fdas_volume_convolve(v, ctypes.c_void_p(spectrum_ptr), ctypes.c_void_p(volume_ptr), ctypes.c_void_p(stream))


def fdas_volume_peaks(v, volume_ptr, threshold, peaks_ptr, capacity, count_ptr, stream=0):
    return lib().fdas_volume_peaks(v, ctypes.c_void_p(volume_ptr), float(threshold), ctypes.c_void_p(peaks_ptr), int(capacity),
                                   ctypes.c_void_p(count_ptr), ctypes.c_void_p(stream))


def fdas_volume_search(v, spectrum_ptr, volume_ptr, threshold, peaks_ptr, capacity, count_ptr, stream=0):
    return lib().fdas_volume_search(v, ctypes.c_void_p(spectrum_ptr), ctypes.c_void_p(volume_ptr), float(threshold),
                                    ctypes.c_void_p(peaks_ptr), int(capacity), ctypes.c_void_p(count_ptr), ctypes.c_void_p(stream))


def fdas_volume_search_host(v, spectrum_host_ptr, threshold, peaks_host_ptr, capacity, stream=0):
    n = ctypes.c_int(0)
    rc = lib().fdas_volume_search_host(v, ctypes.c_void_p(spectrum_host_ptr), float(threshold), ctypes.c_void_p(peaks_host_ptr),
                                       int(capacity), ctypes.byref(n), ctypes.c_void_p(stream))
    return rc, n.value


def fdas_volume_launch_count(v):
    n = ctypes.c_int64()
    rc = lib().fdas_volume_launch_count(v, ctypes.byref(n))
    return rc, n.value


def fdas_volume_last_cuda_error(v):
    return lib().fdas_volume_last_cuda_error(v)


# ---- convenience wrapper ------------------------------------------------------------------
class Plan:
    """Owns one fdas_plan_t.  Tensors are torch CUDA tensors (device memory and streams are
    torch's; all arithmetic is the library's)."""

    def __init__(self, N: int, zmax: float, dz: float, seglen: int, precision="f32", build: bool = True,
                 stream: Optional[int] = None, algorithm="auto", plane="f32", jerk: float = 0.0):
        prec = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        rc, self._h = fdas_plan_create_jerk(N, zmax, dz, jerk, seglen, prec) if jerk else fdas_plan_create(N, zmax, dz, seglen, prec)
        if rc:
            self._h = None
            raise FdasError(rc, "fdas_plan_create")
        rc, self.info = fdas_plan_info(self._h)
        self._check(rc, "fdas_plan_info")
        self.precision = prec
        algo = ALGORITHMS[algorithm] if isinstance(algorithm, str) else int(algorithm)
        if algo != FDAS_ALGO_AUTO:
            self._check(fdas_set_algorithm(self._h, algo), "fdas_set_algorithm")
        self.plane_format = PLANE_FORMATS[plane] if isinstance(plane, str) else int(plane)
        if self.plane_format != FDAS_PLANE_F32:
            self._check(fdas_set_plane_format(self._h, self.plane_format), "fdas_set_plane_format")
            rc, self.info = fdas_plan_info(self._h)
            self._check(rc, "fdas_plan_info")
        if build:
            self.build_templates(stream)

    def _check(self, rc, where):
        if rc:
            raise FdasError(rc, where, fdas_last_cuda_error(self._h))

    # shape helpers
    @property
    def M(self): return int(self.info.n_bins)
    @property
    def K(self): return int(self.info.n_templates)
    @property
    def S(self): return int(self.info.seglen)

    def z_values(self):
        return [fdas_z_of_index(self._h, k)[1] for k in range(self.K)]

    def plane_dtype(self):
        import torch
        if self.plane_format == FDAS_PLANE_BF16:
            return torch.bfloat16          # the library writes bf16 bit patterns; torch reads them as bfloat16
        return torch.float64 if self.precision == FDAS_F64 else torch.float32

    def harmonic_sum(self, plane, n_harmonics: int, out=None, stream: Optional[int] = None, drift: bool = False):
        """fdas_harmonic_sum: S[k][r] = sum_h P[k0 + h (k - k0)][h r]; drift=True takes the
        largest power of each harmonic's quantisation window (fdas_harmonic_sum_drift)."""
        import torch
        assert plane.is_cuda and plane.is_contiguous() and tuple(plane.shape) == (self.K, self.M)
        assert plane.dtype == self.plane_dtype()
        odt = torch.float64 if self.precision == FDAS_F64 else torch.float32
        if out is None:
            out = torch.empty((self.K, self.M), dtype=odt, device=plane.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == odt and tuple(out.shape) == (self.K, self.M)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        fn = fdas_harmonic_sum_drift if drift else fdas_harmonic_sum
        self._check(fn(self._h, plane.data_ptr(), out.data_ptr(), n_harmonics, stream), "fdas_harmonic_sum")
        return out

    def band_max(self, plane, f_bin: float, n_bands: int, stream: Optional[int] = None):
        """fdas_band_max (Table 3): list of (z_index, r, power), one per harmonic band."""
        import numpy as np
        import torch
        assert plane.is_cuda and plane.is_contiguous() and tuple(plane.shape) == (self.K, self.M)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        buf = torch.empty(3 * n_bands, dtype=torch.int32, device=plane.device)
        self._check(fdas_band_max(self._h, plane.data_ptr(), f_bin, n_bands, buf.data_ptr(), stream), "fdas_band_max")
        raw = buf.cpu().numpy().reshape(n_bands, 3)
        return [(int(a), int(b), float(np.int32(c).view(np.float32))) for a, b, c in raw]

    def quick_cast(self, plane_bf16, out=None, stream: Optional[int] = None):
        """fdas_quick_cast: bf16-stored plane(s) -> float32 by byte placement."""
        import torch
        assert plane_bf16.is_cuda and plane_bf16.is_contiguous() and plane_bf16.dtype == torch.bfloat16
        assert tuple(plane_bf16.shape[-2:]) == (self.K, self.M)
        batch = 1 if plane_bf16.dim() == 2 else plane_bf16.shape[0]
        if out is None:
            out = torch.empty(plane_bf16.shape, dtype=torch.float32, device=plane_bf16.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float32 and out.shape == plane_bf16.shape
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._check(fdas_quick_cast(self._h, plane_bf16.data_ptr(), out.data_ptr(), batch, stream), "fdas_quick_cast")
        return out

    def spectrum_dtype(self):
        import torch
        return torch.complex128 if self.precision == FDAS_F64 else torch.complex64

    def spectrum(self, timeseries, out=None, stream: Optional[int] = None):
        """fdas_spectrum: float32 CUDA tensor [N] -> complex spectrum [M] (the real FFT of PAPER.md:85)."""
        import torch
        assert timeseries.is_cuda and timeseries.is_contiguous() and timeseries.dtype == torch.float32
        assert timeseries.numel() == 2 * self.M
        if out is None:
            out = torch.empty(self.M, dtype=self.spectrum_dtype(), device=timeseries.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == self.spectrum_dtype() and out.numel() == self.M
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._check(fdas_spectrum(self._h, timeseries.data_ptr(), out.data_ptr(), stream), "fdas_spectrum")
        return out

    def build_templates(self, stream: Optional[int] = None):
        """Enqueued on torch's current stream unless one is given, like every other call: the build must
        precede fdas_convolve in stream order (include/fdas.h)."""
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        self._check(fdas_build_templates(self._h, stream), "fdas_build_templates")

    def convolve(self, spectrum, plane=None, stream: Optional[int] = None):
        """spectrum: CUDA tensor [M] (or [B, M]) complex64/complex128; returns plane [K, M] ([B, K, M])."""
        import torch
        assert spectrum.is_cuda and spectrum.is_contiguous() and spectrum.dtype == self.spectrum_dtype()
        batch = 1 if spectrum.dim() == 1 else spectrum.shape[0]
        assert spectrum.shape[-1] == self.M
        shape = (self.K, self.M) if spectrum.dim() == 1 else (batch, self.K, self.M)
        if plane is None:
            plane = torch.empty(shape, dtype=self.plane_dtype(), device=spectrum.device)
        assert plane.is_cuda and plane.is_contiguous() and tuple(plane.shape) == shape and plane.dtype == self.plane_dtype()
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._check(fdas_convolve_batched(self._h, spectrum.data_ptr(), plane.data_ptr(), batch, stream),
                    "fdas_convolve")
        return plane

    def peaks(self, plane, threshold: float, capacity: int = 1 << 16, stream: Optional[int] = None):
        """Returns (total_count, records) with records a numpy structured array (z_index, r, power)."""
        import numpy as np
        import torch
        assert plane.is_cuda and plane.is_contiguous() and tuple(plane.shape) == (self.K, self.M)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        buf = torch.empty(max(capacity, 1) * 3, dtype=torch.int32, device=plane.device)
        cnt = torch.zeros(1, dtype=torch.int32, device=plane.device)
        self._check(fdas_peaks(self._h, plane.data_ptr(), threshold, buf.data_ptr() if capacity else 0, capacity,
                               cnt.data_ptr(), stream), "fdas_peaks")
        n = int(cnt.item())
        w = min(n, capacity)
        raw = buf[: 3 * w].cpu().numpy().reshape(w, 3)
        rec = np.zeros(w, dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
        rec["z_index"] = raw[:, 0]
        rec["r"] = raw[:, 1]
        rec["power"] = raw[:, 2].copy().view(np.float32)
        return n, rec

    def search(self, spectrum, threshold: float, plane=None, capacity: int = 1 << 16, stream: Optional[int] = None,
               plane_free: bool = False):
        """fdas_search: returns (plane, total_count, records); plane_free=True passes a NULL plane (returns None for it)."""
        import numpy as np
        import torch
        assert spectrum.is_cuda and spectrum.is_contiguous() and spectrum.dtype == self.spectrum_dtype()
        assert tuple(spectrum.shape) == (self.M,)
        if plane is None and not plane_free:
            plane = torch.empty((self.K, self.M), dtype=self.plane_dtype(), device=spectrum.device)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        buf = torch.empty(max(capacity, 1) * 3, dtype=torch.int32, device=spectrum.device)
        cnt = torch.zeros(1, dtype=torch.int32, device=spectrum.device)
        self._check(fdas_search(self._h, spectrum.data_ptr(), 0 if plane_free else plane.data_ptr(), threshold,
                                buf.data_ptr() if capacity else 0, capacity, cnt.data_ptr(), stream), "fdas_search")
        n = int(cnt.item())
        w = min(n, capacity)
        raw = buf[: 3 * w].cpu().numpy().reshape(w, 3)
        rec = np.zeros(w, dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
        rec["z_index"] = raw[:, 0]
        rec["r"] = raw[:, 1]
        rec["power"] = raw[:, 2].copy().view(np.float32)
        return plane, n, rec

    def search_static(self, spectrum, threshold: float, peaks_buf, count_buf, capacity: int, stream: Optional[int] = None):
        """fdas_search_static: the plane-free search with the library's built-in scratch array; the call allocates
        nothing, so the caller brings the outputs: peaks_buf int32 [3 * capacity], count_buf int32 [1], on the device."""
        import torch
        assert spectrum.is_cuda and spectrum.is_contiguous() and spectrum.dtype == self.spectrum_dtype()
        assert tuple(spectrum.shape) == (self.M,)
        assert peaks_buf.is_cuda and peaks_buf.dtype == torch.int32 and peaks_buf.numel() >= 3 * capacity
        assert count_buf.is_cuda and count_buf.dtype == torch.int32 and count_buf.numel() >= 1
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._check(fdas_search_static(self._h, spectrum.data_ptr(), threshold, peaks_buf.data_ptr() if capacity else 0,
                                       capacity, count_buf.data_ptr(), stream), "fdas_search_static")

    def search_batched(self, spectra, threshold: float, capacity: int = 4096, planes=None, stream: Optional[int] = None):
        """fdas_search_batched: spectra [B, M] on the device; planes [B, K, M] or None (plane-free form).
        Returns (counts [B] numpy, records [B, capacity] numpy structured array; series b's first
        min(counts[b], capacity) records are valid)."""
        import numpy as np
        import torch
        assert spectra.is_cuda and spectra.is_contiguous() and spectra.dtype == self.spectrum_dtype()
        assert spectra.dim() == 2 and spectra.shape[1] == self.M
        B = int(spectra.shape[0])
        if planes is not None:
            assert planes.is_cuda and planes.is_contiguous() and tuple(planes.shape) == (B, self.K, self.M)
            assert planes.dtype == self.plane_dtype()
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        buf = torch.empty((B, max(capacity, 1), 3), dtype=torch.int32, device=spectra.device)
        cnt = torch.zeros(B, dtype=torch.int32, device=spectra.device)
        self._check(fdas_search_batched(self._h, spectra.data_ptr(), 0 if planes is None else planes.data_ptr(), B, threshold,
                                        buf.data_ptr() if capacity else 0, capacity, cnt.data_ptr(), stream),
                    "fdas_search_batched")
        raw = buf.cpu().numpy()
        rec = np.zeros((B, max(capacity, 1)), dtype=[("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
        rec["z_index"] = raw[..., 0]
        rec["r"] = raw[..., 1]
        rec["power"] = raw[..., 2].copy().view(np.float32)
        return cnt.cpu().numpy(), rec

    def convolve_host(self, spectrum_host, plane_host, stream: Optional[int] = None):
        """numpy or pinned torch CPU buffers; copies are inside the call."""
        stream = _current_stream(stream)
        self._check(fdas_convolve_host(self._h, _host_ptr(spectrum_host), _host_ptr(plane_host), stream),
                    "fdas_convolve_host")
        return plane_host

    def search_host(self, spectrum_host, threshold: float, peaks_host, capacity: int, stream: Optional[int] = None):
        stream = _current_stream(stream)
        rc, n = fdas_search_host(self._h, _host_ptr(spectrum_host), threshold, _host_ptr(peaks_host), capacity, stream)
        self._check(rc, "fdas_search_host")
        return n

    def search_host_batched(self, spectra_host, threshold: float, peaks_host, counts_host, capacity: int,
                            stream: Optional[int] = None, timeseries: bool = False):
        """spectra_host [B, M] (timeseries=True: the fp32 series [B, N]); peaks_host >= B*capacity records (12 bytes each);
        counts_host [B] int32 (numpy or pinned torch)."""
        stream = _current_stream(stream)
        n = int(spectra_host.shape[0])
        fn = fdas_search_host_timeseries_batched if timeseries else fdas_search_host_batched
        self._check(fn(self._h, _host_ptr(spectra_host), n, threshold, _host_ptr(peaks_host), capacity,
                       _host_ptr(counts_host), stream), "fdas_search_host_batched")
        return counts_host

    def search_host_timeseries(self, timeseries_host, threshold: float, peaks_host, capacity: int, stream: Optional[int] = None):
        """fdas_search_host_timeseries: fp32 series [N] on the host in, peak list out (real FFT and search on the device)."""
        stream = _current_stream(stream)
        rc, n = fdas_search_host_timeseries(self._h, _host_ptr(timeseries_host), threshold, _host_ptr(peaks_host), capacity, stream)
        self._check(rc, "fdas_search_host_timeseries")
        return n

    def templates(self):
        """Bank in natural order as numpy: complex128/complex64, or uint16 [K, S, 2] bit patterns for bf16."""
        import numpy as np
        if self.precision == FDAS_F64:
            out = np.empty((self.K, self.S), dtype=np.complex128)
        elif self.precision == FDAS_F32:
            out = np.empty((self.K, self.S), dtype=np.complex64)
        else:
            out = np.empty((self.K, self.S, 2), dtype=np.uint16)
        self._check(fdas_templates_host(self._h, out.ctypes.data, out.nbytes), "fdas_templates_host")
        return out

    def taps(self):
        import numpy as np
        m = int(self.info.halfwidth_max)
        out = np.empty((self.K, 2 * m + 1), dtype=np.complex128)
        self._check(fdas_taps_host(self._h, out.ctypes.data, out.nbytes), "fdas_taps_host")
        return out

    def tapmatrix(self):
        """bf16 plans: the taps the tensor-core path uses, uint16 bit patterns [K, 2*m_max+1, 2]."""
        import numpy as np
        m = int(self.info.halfwidth_max)
        out = np.empty((self.K, 2 * m + 1, 2), dtype=np.uint16)
        self._check(fdas_tapmatrix_host(self._h, out.ctypes.data, out.nbytes), "fdas_tapmatrix_host")
        return out

    def algorithm(self) -> str:
        rc, a = fdas_get_algorithm(self._h)
        self._check(rc, "fdas_get_algorithm")
        return {FDAS_ALGO_FFT: "fft", FDAS_ALGO_MMA: "mma", FDAS_ALGO_MMA_SCALAR: "mma_scalar"}[a]

    def describe(self, plane=None, batch: int = 1) -> dict:
        """fdas_describe_convolve as a dict: the kernel fdas_convolve would launch for this plane buffer (None: the scan
        launch of the plane-free search), its grid and the tensor flops it issues."""
        rc, info = fdas_describe_convolve(self._h, 0 if plane is None else plane.data_ptr(), batch)
        self._check(rc, "fdas_describe_convolve")
        d = {name: getattr(info, name) for name, _ in info._fields_}
        d["kernel"] = info.kernel.decode()
        d["algorithm"] = {FDAS_ALGO_FFT: "fft", FDAS_ALGO_MMA: "mma", FDAS_ALGO_MMA_SCALAR: "mma_scalar"}[info.algorithm]
        return d

    def launch_count(self) -> int:
        return fdas_launch_count(self._h)[1]

    def close(self):
        if getattr(self, "_h", None):
            fdas_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Volume:
    """Owns one fdas_volume_t (the f-fdot-fddot volume of a jerk search): slabs w_i = -wmax + i dw."""

    def __init__(self, N: int, zmax: float, dz: float, wmax: float, dw: float, seglen: int, precision="f32",
                 algorithm="auto", stream: Optional[int] = None):
        prec = PRECISIONS[precision] if isinstance(precision, str) else int(precision)
        rc, self._v = fdas_volume_create(N, zmax, dz, wmax, dw, seglen, prec)
        if rc:
            self._v = None
            raise FdasError(rc, "fdas_volume_create")
        self.precision = prec
        rc, self.info = fdas_volume_info(self._v)
        self._check(rc, "fdas_volume_info")
        algo = ALGORITHMS[algorithm] if isinstance(algorithm, str) else int(algorithm)
        if algo != FDAS_ALGO_AUTO:
            self._check(fdas_volume_set_algorithm(self._v, algo), "fdas_volume_set_algorithm")
        self._check(fdas_volume_build_templates(self._v, _current_stream(stream)), "fdas_volume_build_templates")

    def _check(self, rc, where):
        if rc:
            raise FdasError(rc, where, fdas_volume_last_cuda_error(self._v))

    @property
    def W(self): return int(self.info.n_slabs)
    @property
    def K(self): return int(self.info.n_templates)
    @property
    def M(self): return int(self.info.n_bins)

    def w_values(self):
        return [fdas_volume_w_of_index(self._v, i)[1] for i in range(self.W)]

    def dtype(self):
        import torch
        return torch.float64 if self.precision == FDAS_F64 else torch.float32

    def convolve(self, spectrum, volume=None, stream: Optional[int] = None):
        import torch
        assert spectrum.is_cuda and spectrum.is_contiguous() and tuple(spectrum.shape) == (self.M,)
        if volume is None:
            volume = torch.empty((self.W, self.K, self.M), dtype=self.dtype(), device=spectrum.device)
        assert volume.is_cuda and volume.is_contiguous() and tuple(volume.shape) == (self.W, self.K, self.M) and volume.dtype == self.dtype()
        self._check(fdas_volume_convolve(self._v, spectrum.data_ptr(), volume.data_ptr(), _current_stream(stream)), "fdas_volume_convolve")
        return volume

    @staticmethod
    def _records(buf, n, capacity):
        import numpy as np
        w = min(n, capacity)
        raw = buf[: 4 * w].cpu().numpy().reshape(w, 4)
        rec = np.zeros(w, dtype=[("w_index", np.int32), ("z_index", np.int32), ("r", np.int32), ("power", np.float32)])
        rec["w_index"], rec["z_index"], rec["r"] = raw[:, 0], raw[:, 1], raw[:, 2]
        rec["power"] = raw[:, 3].copy().view(np.float32)
        return rec

    def peaks(self, volume, threshold: float, capacity: int = 1 << 16, stream: Optional[int] = None):
        """fdas_volume_peaks: returns (total_count, records (w_index, z_index, r, power))."""
        import torch
        assert volume.is_cuda and volume.is_contiguous() and tuple(volume.shape) == (self.W, self.K, self.M)
        buf = torch.empty(max(capacity, 1) * 4, dtype=torch.int32, device=volume.device)
        cnt = torch.zeros(1, dtype=torch.int32, device=volume.device)
        self._check(fdas_volume_peaks(self._v, volume.data_ptr(), threshold, buf.data_ptr() if capacity else 0, capacity,
                                      cnt.data_ptr(), _current_stream(stream)), "fdas_volume_peaks")
        n = int(cnt.item())
        return n, self._records(buf, n, capacity)

    def search(self, spectrum, threshold: float, volume=None, capacity: int = 1 << 16, stream: Optional[int] = None):
        """fdas_volume_search: returns (volume, total_count, records)."""
        import torch
        assert spectrum.is_cuda and spectrum.is_contiguous() and tuple(spectrum.shape) == (self.M,)
        if volume is None:
            volume = torch.empty((self.W, self.K, self.M), dtype=self.dtype(), device=spectrum.device)
        buf = torch.empty(max(capacity, 1) * 4, dtype=torch.int32, device=spectrum.device)
        cnt = torch.zeros(1, dtype=torch.int32, device=spectrum.device)
        self._check(fdas_volume_search(self._v, spectrum.data_ptr(), volume.data_ptr(), threshold, buf.data_ptr() if capacity else 0,
                                       capacity, cnt.data_ptr(), _current_stream(stream)), "fdas_volume_search")
        n = int(cnt.item())
        return volume, n, self._records(buf, n, capacity)

    def search_host(self, spectrum_host, threshold: float, peaks_host, capacity: int, stream: Optional[int] = None):
        rc, n = fdas_volume_search_host(self._v, _host_ptr(spectrum_host), threshold, _host_ptr(peaks_host), capacity, _current_stream(stream))
        self._check(rc, "fdas_volume_search_host")
        return n

    def launch_count(self) -> int:
        return fdas_volume_launch_count(self._v)[1]

    def close(self):
        if getattr(self, "_v", None):
            fdas_volume_destroy(self._v)
            self._v = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _current_stream(stream: Optional[int]) -> int:
    """torch's current stream when the caller names none (the stream the templates were built on by default)."""
    if stream is not None:
        return stream
    import torch
    return torch.cuda.current_stream().cuda_stream


def _host_ptr(buf) -> int:
    if hasattr(buf, "data_ptr"):
        assert not buf.is_cuda
        return buf.data_ptr()
    return buf.ctypes.data
