// fdas_plan.cu -- plan lifetime, argument checking and the C-ABI entry points of libfdas.
// Every entry point is documented in include/fdas.h.
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <vector>
#include "fdas_internal.h"

// m = ceil(|z|/2 + |w|/12) + 16: the largest excursion of the frequency from its mean, plus 16 bins (w = 0: BASELINE.json's rule)
static int halfwidth_of(double z, double w) { return (int)ceil(fabs(z) / 2.0 + fabs(w) / 12.0) + 16; }

static void free_device_members(fdas_plan *p)
{
    cudaFree(p->bank);
    cudaFree(p->taps);
    cudaFree(p->twiddle);
    cudaFree(p->band_scratch);
    cudaFree(p->rfft_scratch);
    if (p->pipe_ready) {
        cudaStreamDestroy(p->pipe_stream);
        cudaStreamDestroy(p->pipe_stream_back);
        for (int e = 0; e < 3; ++e)
            for (int b = 0; b < 2; ++b) cudaEventDestroy(p->pipe_ev[e][b]);
        for (int c = 0; c < 6; ++c) cudaEventDestroy(p->chunk_ev[c]);
    }
    for (int b = 0; b < 2; ++b) {
        cudaFree(p->pipe_spec[b]);
        cudaFree(p->pipe_series[b]);
        cudaFree(p->pipe_peaks[b]);
        cudaFree(p->pipe_count[b]);
    }
    cudaFree(p->tc_bmat);
    cudaFree(p->tc_ktab);
    cudaFree(p->tc_kref);
    cudaFree(p->tc_ranges);
    free(p->tc_maps);
    cudaFree(p->cand);
    cudaFree(p->cand_ctr);
    cudaFree(p->tf_flags);
    cudaFree(p->tf_list);
    cudaFree(p->tf_ctr);
    cudaFree(p->tf_scratch);
    free(p->tf_maps);
    cudaFree(p->stage_spectrum);
    cudaFree(p->stage_series);
    cudaFree(p->stage_plane);
    cudaFree(p->stage_peaks);
    cudaFree(p->stage_count);
    cudaFreeHost(p->host_tail);
}

extern "C" int fdas_plan_create(fdas_plan_t **out, int64_t N, double zmax, double dz, int seglen,
                                int precision)
{
    return fdas_plan_create_jerk(out, N, zmax, dz, 0.0, seglen, precision);
}

extern "C" int fdas_plan_create_jerk(fdas_plan_t **out, int64_t N, double zmax, double dz, double w, int seglen,
                                     int precision)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    *out = NULL;
    if (!(zmax >= 0.0) || !(dz > 0.0) || !isfinite(zmax) || !isfinite(dz) || !isfinite(w)) return FDAS_ERR_INVALID_ARG;
    if (precision != FDAS_F64 && precision != FDAS_F32 && precision != FDAS_BF16) return FDAS_ERR_INVALID_ARG;
    if (seglen == 8192) return FDAS_ERR_UNSUPPORTED;
    if (seglen != 256 && seglen != 512 && seglen != 1024 && seglen != 2048 && seglen != 4096)
        return FDAS_ERR_INVALID_ARG;
    if (N < 2 * (int64_t)seglen || (N & 1)) return FDAS_ERR_INVALID_ARG;
    double kk = floor(zmax / dz + 1e-9);
    if (kk > 2047.0) return FDAS_ERR_INVALID_ARG;
    const int K = 2 * (int)kk + 1;
    const int m_max = halfwidth_of(zmax, w);
    const int L = (m_max + 31) / 32 * 32;
    const int V = (seglen - L - m_max) / 32 * 32;
    if (V < 32) return FDAS_ERR_INVALID_ARG;

    fdas_plan *p = new (std::nothrow) fdas_plan;
    if (!p) return FDAS_ERR_ALLOC;
    memset(p, 0, sizeof(*p));
    p->N = N;
    p->M = N / 2;
    p->zmax = zmax;
    p->dz = dz;
    p->jerk = w;
    p->K = K;
    p->S = seglen;
    p->m_max = m_max;
    p->L = L;
    p->V = V;
    p->precision = precision;
    p->n_seg = (p->M + V - 1) / V;
    p->T = seglen / FDAS_PTS;
    p->R3 = seglen / 256;
    p->last_err = cudaSuccess;

    cudaError_t e = cudaGetDevice(&p->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, p->device);
    if (e != cudaSuccess) {
        delete p;
        return FDAS_ERR_CUDA;
    }
    p->bank_bytes = (size_t)K * seglen * 2 * fdas_storage_scalar_bytes(precision);
    const size_t tw_bytes = (size_t)seglen * (precision == FDAS_F64 ? sizeof(double2) : sizeof(float2));
    const size_t taps_bytes = (size_t)K * (2 * m_max + 1) * sizeof(double2);
    if ((e = cudaMalloc(&p->bank, p->bank_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->taps, taps_bytes)) != cudaSuccess ||
        (e = cudaMalloc(&p->twiddle, tw_bytes)) != cudaSuccess) {
        free_device_members(p);
        delete p;
        cudaGetLastError();
        return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
    }
    const int rc = fdas_mma_plan(p);
    if (rc != FDAS_OK) {
        free_device_members(p);
        delete p;
        cudaGetLastError();
        return rc;
    }
    *out = p;
    return FDAS_OK;
}

extern "C" int fdas_set_algorithm(fdas_plan_t *p, int algorithm)
{
    if (!p) return FDAS_ERR_INVALID_ARG;
    if (algorithm != FDAS_ALGO_AUTO && algorithm != FDAS_ALGO_FFT && algorithm != FDAS_ALGO_MMA &&
        algorithm != FDAS_ALGO_MMA_SCALAR)
        return FDAS_ERR_INVALID_ARG;
    const bool mma = algorithm == FDAS_ALGO_MMA || algorithm == FDAS_ALGO_MMA_SCALAR;
    if (mma && !((p->precision == FDAS_BF16 || (p->precision == FDAS_F32 && p->M % 4 == 0 && algorithm == FDAS_ALGO_MMA)) && p->tc_supported))
        return FDAS_ERR_UNSUPPORTED;
    if (algorithm == FDAS_ALGO_FFT && p->plane_bf16) return FDAS_ERR_UNSUPPORTED;   // only the tensor-core kernels write a bf16 plane
    p->algo = mma ? FDAS_ALGO_MMA : algorithm;
    p->tc_force_scalar_stores = algorithm == FDAS_ALGO_MMA_SCALAR;
    return FDAS_OK;
}

extern "C" int fdas_get_algorithm(const fdas_plan_t *p, int *algorithm)
{
    if (!p || !algorithm) return FDAS_ERR_INVALID_ARG;
    *algorithm = fdas_uses_mma(p) ? ((p->tc_force_scalar_stores || (p->M * fdas_plane_elem_bytes(p)) % 16 != 0) ? FDAS_ALGO_MMA_SCALAR : FDAS_ALGO_MMA)
                                  : FDAS_ALGO_FFT;
    return FDAS_OK;
}

extern "C" int fdas_set_plane_format(fdas_plan_t *p, int format)
{
    if (!p) return FDAS_ERR_INVALID_ARG;
    if (format != FDAS_PLANE_F32 && format != FDAS_PLANE_BF16) return FDAS_ERR_INVALID_ARG;
    // a bf16 plane is written by the tensor-core kernels only
    if (format == FDAS_PLANE_BF16 && !(p->precision == FDAS_BF16 && fdas_uses_mma(p))) return FDAS_ERR_UNSUPPORTED;
    if (p->plane_bf16 != (format == FDAS_PLANE_BF16)) {   // the host-path staging plane has the old element size
        cudaFree(p->stage_plane);
        p->stage_plane = NULL;
    }
    p->plane_bf16 = format == FDAS_PLANE_BF16;
    return FDAS_OK;
}

extern "C" int fdas_get_plane_format(const fdas_plan_t *p, int *format)
{
    if (!p || !format) return FDAS_ERR_INVALID_ARG;
    *format = p->plane_bf16 ? FDAS_PLANE_BF16 : FDAS_PLANE_F32;
    return FDAS_OK;
}

extern "C" int fdas_quick_cast(fdas_plan_t *p, const void *plane_bf16_dev, void *plane_f32_dev, int batch, void *stream)
{
    if (!p || !plane_bf16_dev || !plane_f32_dev || batch < 1) return FDAS_ERR_INVALID_ARG;
    return fdas_launch_quick_cast(p, plane_bf16_dev, plane_f32_dev, (long long)batch * p->K * p->M, (cudaStream_t)stream);
}

static int harmonic_sum_common(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, int drift, void *stream);

extern "C" int fdas_harmonic_sum(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, void *stream)
{
    return harmonic_sum_common(p, plane_dev, sum_dev, n_harmonics, 0, stream);
}

extern "C" int fdas_harmonic_sum_drift(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, void *stream)
{
    return harmonic_sum_common(p, plane_dev, sum_dev, n_harmonics, 1, stream);
}

static int harmonic_sum_common(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, int drift, void *stream)
{
    if (!p || !plane_dev || !sum_dev || n_harmonics < 1 || n_harmonics > 32) return FDAS_ERR_INVALID_ARG;
    // harmonic h of row z_k is row z = h z_k: on the grid iff z = 0 is (zmax a multiple of dz)
    const int k0 = (p->K - 1) / 2;
    if (fabs(-p->zmax + k0 * p->dz) > 1e-9 * (1.0 + p->zmax)) return FDAS_ERR_UNSUPPORTED;
    return fdas_launch_harmonic_sum(p, plane_dev, sum_dev, n_harmonics, k0, drift, (cudaStream_t)stream);
}

extern "C" int fdas_spectrum(fdas_plan_t *p, const void *timeseries_dev, void *spectrum_dev, void *stream)
{
    if (!p || !timeseries_dev || !spectrum_dev) return FDAS_ERR_INVALID_ARG;
    return fdas_launch_spectrum(p, timeseries_dev, spectrum_dev, (cudaStream_t)stream);
}

extern "C" int fdas_band_max(fdas_plan_t *p, const void *plane_dev, double f_bin, int n_bands, fdas_peak_t *out_dev, void *stream)
{
    if (!p || !plane_dev || !out_dev || n_bands < 1 || n_bands > FDAS_MAX_BANDS || !(f_bin > 0.0) || !(f_bin < 1e15))
        return FDAS_ERR_INVALID_ARG;
    return fdas_launch_band_max(p, plane_dev, f_bin, n_bands, out_dev, (cudaStream_t)stream);
}

extern "C" int fdas_plan_destroy(fdas_plan_t *p)
{
    if (!p) return FDAS_OK;
    cudaDeviceSynchronize();
    free_device_members(p);
    delete p;
    return FDAS_OK;
}

extern "C" int fdas_plan_info(const fdas_plan_t *p, fdas_info_t *info)
{
    if (!p || !info) return FDAS_ERR_INVALID_ARG;
    info->n_bins = p->M;
    info->n_templates = p->K;
    info->seglen = p->S;
    info->halfwidth_max = p->m_max;
    info->overlap_left = p->L;
    info->valid_per_seg = p->V;
    info->precision = p->precision;
    info->n_segments = p->n_seg;
    info->plane_row_pitch = p->M;
    info->plane_elem_bytes = fdas_plane_elem_bytes(p);
    info->spectrum_elem_bytes = p->precision == FDAS_F64 ? 16 : 8;
    info->bank_bytes = p->bank_bytes;
    return FDAS_OK;
}

extern "C" int fdas_z_of_index(const fdas_plan_t *p, int k, double *z)
{
    if (!p || !z || k < 0 || k >= p->K) return FDAS_ERR_INVALID_ARG;
    *z = -p->zmax + k * p->dz;
    return FDAS_OK;
}

extern "C" int fdas_build_templates(fdas_plan_t *p, void *stream)
{
    if (!p) return FDAS_ERR_INVALID_ARG;
    int rc = fdas_launch_build_templates(p, (cudaStream_t)stream);
    if (rc == FDAS_OK) rc = fdas_launch_build_tapmatrix(p, (cudaStream_t)stream);
    if (rc == FDAS_OK) p->built = 1;
    return rc;
}

extern "C" int fdas_convolve_batched(fdas_plan_t *p, const void *spectra_dev, void *planes_dev,
                                     int batch, void *stream)
{
    if (!p || !spectra_dev || !planes_dev || batch < 1) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    return fdas_launch_convolve(p, spectra_dev, planes_dev, batch, (cudaStream_t)stream);
}

extern "C" int fdas_convolve(fdas_plan_t *p, const void *spectrum_dev, void *plane_dev, void *stream)
{
    return fdas_convolve_batched(p, spectrum_dev, plane_dev, 1, stream);
}

extern "C" int fdas_peaks(fdas_plan_t *p, const void *plane_dev, float threshold,
                          fdas_peak_t *peaks_dev, int capacity, int *count_dev, void *stream)
{
    if (!p || !plane_dev || !count_dev || capacity < 0 || (capacity > 0 && !peaks_dev))
        return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    return fdas_launch_peaks(p, plane_dev, threshold, peaks_dev, capacity, count_dev,
                             (cudaStream_t)stream);
}

// The arguments of a convolve launch with the fused threshold test (fdas_search, fdas_volume_search): the plan's
// candidate buffer and its two counters, used alternately from call to call.
int fdas_search_prepare(fdas_plan *p, float thr, int *count_dev, cudaStream_t st, fdas_search_args *sa)
{
    *sa = fdas_search_args{};
    if (!p->cand || !p->cand_ctr) {   // both or neither: a failed second allocation must not leave a NULL counter behind
        cudaFree(p->cand);
        cudaFree(p->cand_ctr);
        p->cand = NULL;
        p->cand_ctr = NULL;
        p->cand_capacity = 1 << 18;
        fdas_peak_t *c = NULL;
        int *ctr = NULL;
        cudaError_t e = cudaMalloc((void **)&c, sizeof(fdas_peak_t) * (size_t)p->cand_capacity);
        if (e == cudaSuccess) e = cudaMalloc((void **)&ctr, 2 * sizeof(int));
        if (e == cudaSuccess) e = cudaMemsetAsync(ctr, 0, 2 * sizeof(int), st);
        if (e != cudaSuccess) {
            cudaFree(c);
            cudaFree(ctr);
            p->last_err = e;
            return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
        }
        p->cand = c;
        p->cand_ctr = ctr;
    }
    sa->enabled = 1;
    sa->thr = thr;
    sa->cand = p->cand;
    sa->cand_count = p->cand_ctr + (p->search_calls & 1);
    sa->cand_count_next = p->cand_ctr + ((p->search_calls + 1) & 1);
    sa->cand_capacity = p->cand_capacity;
    sa->count_out = count_dev;
    sa->cand_span = 8;   // overwritten by the convolve launch
    p->search_calls += 1;
    return FDAS_OK;
}

// fdas_search: convolve + peaks.  On the tensor-core path the convolve epilogue flags the
// (rare) chunks holding a power above the threshold and a small second kernel applies the
// peak rule to those cells only, so the plane is not read back from HBM.
static int search_on_device(fdas_plan *p, const void *spectrum_dev, void *plane_dev, float threshold,
                            fdas_peak_t *peaks_dev, int capacity, int *count_dev, cudaStream_t st)
{
    if (!plane_dev)   // plane-free form: scan launch + recheck launch (fdas_mma_search.cu)
        return fdas_launch_search_noplane(p, spectrum_dev, 1, threshold, peaks_dev, capacity, count_dev, st);
    if (!fdas_uses_mma(p)) {
        // overlap-save FFT forms: the store loop lists the cells above the threshold, a small launch resolves them
        fdas_search_args sa;
        int rc = fdas_search_prepare(p, threshold, count_dev, st, &sa);
        if (rc) return rc;
        rc = fdas_launch_convolve_fft_search(p, spectrum_dev, plane_dev, &sa, st);
        if (rc) return rc;
        return fdas_launch_resolve_cells(p, plane_dev, sa, peaks_dev, capacity, st);
    }
    fdas_search_args sa;
    { const int rc0 = fdas_search_prepare(p, threshold, count_dev, st, &sa); if (rc0) return rc0; }
    int rc = fdas_launch_convolve_mma(p, spectrum_dev, plane_dev, 1, st, &sa);   // sets sa.cand_span
    if (rc == FDAS_ERR_UNSUPPORTED && p->precision == FDAS_F32 && p->algo == FDAS_ALGO_AUTO) {
        // the split-operand kernel cannot take this plane buffer (alignment, shared memory): FFT kernel + peak pass
        p->search_calls -= 1;
        rc = fdas_launch_convolve(p, spectrum_dev, plane_dev, 1, st);
        if (rc) return rc;
        return fdas_launch_peaks(p, plane_dev, threshold, peaks_dev, capacity, count_dev, st);
    }
    if (rc) return rc;
    return fdas_launch_resolve(p, plane_dev, sa, peaks_dev, capacity, st);
}

extern "C" int fdas_search(fdas_plan_t *p, const void *spectrum_dev, void *plane_dev, float threshold,
                           fdas_peak_t *peaks_dev, int capacity, int *count_dev, void *stream)
{
    if (!p || !spectrum_dev || !count_dev || capacity < 0 || (capacity > 0 && !peaks_dev))
        return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    return search_on_device(p, spectrum_dev, plane_dev, threshold, peaks_dev, capacity, count_dev,
                            (cudaStream_t)stream);
}

extern "C" int fdas_search_batched(fdas_plan_t *p, const void *spectra_dev, void *planes_dev, int batch, float threshold,
                                   fdas_peak_t *peaks_dev, int capacity, int *counts_dev, void *stream)
{
    if (!p || !spectra_dev || !counts_dev || batch < 1 || capacity < 0 || (capacity > 0 && !peaks_dev))
        return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    if (!planes_dev)   // one scan launch and one recheck launch for the whole batch
        return fdas_launch_search_noplane(p, spectra_dev, batch, threshold, peaks_dev, capacity, counts_dev, st);
    const size_t spec_bytes = (size_t)p->M * (p->precision == FDAS_F64 ? 16 : 8);
    const size_t plane_bytes = (size_t)p->K * p->M * fdas_plane_elem_bytes(p);
    for (int b = 0; b < batch; ++b) {
        const int rc = search_on_device(p, static_cast<const unsigned char *>(spectra_dev) + (size_t)b * spec_bytes,
                                        static_cast<unsigned char *>(planes_dev) + (size_t)b * plane_bytes, threshold,
                                        peaks_dev + (size_t)b * capacity, capacity, counts_dev + b, st);
        if (rc) return rc;
    }
    return FDAS_OK;
}

// true when fdas_search can run without a plane for this plan (fdas_launch_search_noplane's own test)
static bool search_is_plane_free(const fdas_plan *p)
{
    return fdas_uses_mma(p) && !p->plane_bf16 && p->tc_bulk_ok && p->tc_groups <= 8;
}

static int ensure_staging(fdas_plan *p, bool want_plane, int peaks_capacity)
{
    const size_t spec_bytes = (size_t)p->M * (p->precision == FDAS_F64 ? 16 : 8);
    const size_t plane_bytes = (size_t)p->K * p->M * fdas_plane_elem_bytes(p);
    if (!p->stage_spectrum) FDAS_CUDA_TRY(p, cudaMalloc(&p->stage_spectrum, spec_bytes));
    if (want_plane && !p->stage_plane) FDAS_CUDA_TRY(p, cudaMalloc(&p->stage_plane, plane_bytes));
    if (!p->stage_count) FDAS_CUDA_TRY(p, cudaMalloc((void **)&p->stage_count, sizeof(int)));
    if (!p->host_tail) FDAS_CUDA_TRY(p, cudaMallocHost(&p->host_tail, 16 + sizeof(fdas_peak_t) * FDAS_TAIL_PEAKS));
    if (peaks_capacity > p->stage_peaks_capacity) {
        cudaFree(p->stage_peaks);
        p->stage_peaks = NULL;
        p->stage_peaks_capacity = 0;
        FDAS_CUDA_TRY(p, cudaMalloc((void **)&p->stage_peaks, sizeof(fdas_peak_t) * (size_t)peaks_capacity));
        p->stage_peaks_capacity = peaks_capacity;
    }
    return FDAS_OK;
}

extern "C" int fdas_convolve_host(fdas_plan_t *p, const void *spectrum_host, void *plane_host,
                                  void *stream)
{
    if (!p || !spectrum_host || !plane_host) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ensure_staging(p, true, 0);
    if (rc) return rc;
    const size_t spec_bytes = (size_t)p->M * (p->precision == FDAS_F64 ? 16 : 8);
    const size_t plane_bytes = (size_t)p->K * p->M * fdas_plane_elem_bytes(p);
    FDAS_CUDA_TRY(p, cudaMemcpyAsync(p->stage_spectrum, spectrum_host, spec_bytes, cudaMemcpyHostToDevice, st));
    rc = fdas_launch_convolve(p, p->stage_spectrum, p->stage_plane, 1, st);
    if (rc) return rc;
    FDAS_CUDA_TRY(p, cudaMemcpyAsync(plane_host, p->stage_plane, plane_bytes, cudaMemcpyDeviceToHost, st));
    FDAS_CUDA_TRY(p, cudaStreamSynchronize(st));
    return FDAS_OK;
}

// the second stream and the events of the host pipelines
static int ensure_pipe(fdas_plan *p)
{
    if (p->pipe_ready) return FDAS_OK;
    FDAS_CUDA_TRY(p, cudaStreamCreateWithFlags(&p->pipe_stream, cudaStreamNonBlocking));
    FDAS_CUDA_TRY(p, cudaStreamCreateWithFlags(&p->pipe_stream_back, cudaStreamNonBlocking));
    for (int e = 0; e < 3; ++e)
        for (int b = 0; b < 2; ++b) FDAS_CUDA_TRY(p, cudaEventCreateWithFlags(&p->pipe_ev[e][b], cudaEventDisableTiming));
    for (int c = 0; c < 6; ++c) FDAS_CUDA_TRY(p, cudaEventCreateWithFlags(&p->chunk_ev[c], cudaEventDisableTiming));
    p->pipe_ready = 1;
    return FDAS_OK;
}

// host input of the *_host search entry points: the complex spectrum, or (timeseries) the N fp32 samples, which
// fdas_spectrum turns into the spectrum on the device (the accelerated flow of the paper's Fig. 1 starts at the series)
static int search_host_common(fdas_plan_t *p, const void *input_host, bool timeseries, float threshold,
                              fdas_peak_t *peaks_host, int capacity, int *count_host, void *stream)
{
    if (!p || !input_host || !count_host || capacity < 0 || (capacity > 0 && !peaks_host))
        return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    const bool plane_free = search_is_plane_free(p);   // no staging plane then: nothing but the spectrum and the peak list in HBM
    int rc = ensure_staging(p, !plane_free, capacity);
    if (rc) return rc;
    const size_t spec_bytes = (size_t)p->M * (p->precision == FDAS_F64 ? 16 : 8);
    bool chunked = false;
    if (timeseries) {
        const size_t ts_bytes = (size_t)p->N * sizeof(float);
        if (!p->stage_series) FDAS_CUDA_TRY(p, cudaMalloc(&p->stage_series, ts_bytes));
        FDAS_CUDA_TRY(p, cudaMemcpyAsync(p->stage_series, input_host, ts_bytes, cudaMemcpyHostToDevice, st));
        rc = fdas_launch_spectrum(p, p->stage_series, p->stage_spectrum, st);
        if (rc) return rc;
    } else if (plane_free && spec_bytes >= ((size_t)8 << 20)) {
        // The spectrum crosses the host link in chunks on a second stream while the scan launch of the plane-free
        // search works through the chunks already on the device (a chunk's last tiles read the first bins of the next
        // chunk, so chunk c is scanned when chunk c + 1 has landed); one recheck launch at the end.  The copy takes
        // 0.6 ms for config 3, the search 0.19 ms: overlapped, a series costs little more than its copy.
        rc = ensure_pipe(p);
        if (rc) return rc;
        cudaStream_t cs = p->pipe_stream;
        const int R = fdas_noplane_block_bins(p, 1);
        const int blocks = (int)((p->M + R - 1) / R);
        // chunks of 1/2, 1/4, 1/8, 1/16, 1/16 of the blocks: every copy call costs a few us of link time, and only the scan
        // of the LAST chunk is not hidden behind a copy
        int first[6] = {0, blocks / 2, blocks / 2 + blocks / 4, blocks - blocks / 8, blocks - blocks / 16, blocks};
        const int n_chunks = blocks >= 64 ? 5 : 1;
        if (n_chunks == 1) first[1] = blocks;
        const size_t esz = spec_bytes / (size_t)p->M;
        fdas_search_args sa;
        rc = fdas_noplane_begin(p, 1, threshold, p->stage_peaks, capacity, p->stage_count, st, &sa);
        if (rc) return rc;
        FDAS_CUDA_TRY(p, cudaEventRecord(p->chunk_ev[0], st));           // after whatever the caller queued before
        FDAS_CUDA_TRY(p, cudaStreamWaitEvent(cs, p->chunk_ev[0], 0));
        for (int c = 0; c < n_chunks; ++c) {
            const long long b0 = (long long)first[c] * R, b1 = (long long)first[c + 1] * R < p->M ? (long long)first[c + 1] * R : p->M;
            FDAS_CUDA_TRY(p, cudaMemcpyAsync(static_cast<unsigned char *>(p->stage_spectrum) + (size_t)b0 * esz,
                                             static_cast<const unsigned char *>(input_host) + (size_t)b0 * esz,
                                             (size_t)(b1 - b0) * esz, cudaMemcpyHostToDevice, cs));
            FDAS_CUDA_TRY(p, cudaEventRecord(p->chunk_ev[1 + c], cs));
        }
        for (int c = 0; c < n_chunks; ++c) {
            const int need = c + 1 < n_chunks ? c + 1 : c;                   // the chunk holding this range's right halo
            FDAS_CUDA_TRY(p, cudaStreamWaitEvent(st, p->chunk_ev[1 + need], 0));
            rc = fdas_noplane_scan(p, p->stage_spectrum, 1, &sa, first[c], first[c + 1] - first[c], st);
            if (rc) return rc;
        }
        rc = fdas_noplane_recheck(p, p->stage_spectrum, 1, &sa, st);
        if (rc) return rc;
        chunked = true;
    } else {
        FDAS_CUDA_TRY(p, cudaMemcpyAsync(p->stage_spectrum, input_host, spec_bytes, cudaMemcpyHostToDevice, st));
    }
    if (!chunked)
        rc = search_on_device(p, p->stage_spectrum, plane_free ? NULL : p->stage_plane, threshold, p->stage_peaks, capacity,
                              p->stage_count, st);
    if (rc) return rc;
    // the count and the first FDAS_TAIL_PEAKS records come back together into pinned memory of the plan: one
    // synchronisation instead of two for every search that finds no more than that (config 3: ~700 peaks)
    int *const tail_count = static_cast<int *>(p->host_tail);
    fdas_peak_t *const tail_peaks = reinterpret_cast<fdas_peak_t *>(static_cast<unsigned char *>(p->host_tail) + 16);
    const int n_tail = capacity < FDAS_TAIL_PEAKS ? capacity : FDAS_TAIL_PEAKS;
    FDAS_CUDA_TRY(p, cudaMemcpyAsync(tail_count, p->stage_count, sizeof(int), cudaMemcpyDeviceToHost, st));
    if (n_tail > 0)
        FDAS_CUDA_TRY(p, cudaMemcpyAsync(tail_peaks, p->stage_peaks, sizeof(fdas_peak_t) * (size_t)n_tail, cudaMemcpyDeviceToHost, st));
    FDAS_CUDA_TRY(p, cudaStreamSynchronize(st));
    *count_host = *tail_count;
    const int n = *count_host < capacity ? *count_host : capacity;
    if (n > 0 && n <= n_tail) {
        memcpy(peaks_host, tail_peaks, sizeof(fdas_peak_t) * (size_t)n);
    } else if (n > 0) {
        FDAS_CUDA_TRY(p, cudaMemcpyAsync(peaks_host, p->stage_peaks, sizeof(fdas_peak_t) * (size_t)n,
                                         cudaMemcpyDeviceToHost, st));
        FDAS_CUDA_TRY(p, cudaStreamSynchronize(st));
    }
    return FDAS_OK;
}

extern "C" int fdas_search_host(fdas_plan_t *p, const void *spectrum_host, float threshold,
                                fdas_peak_t *peaks_host, int capacity, int *count_host, void *stream)
{
    return search_host_common(p, spectrum_host, false, threshold, peaks_host, capacity, count_host, stream);
}

extern "C" int fdas_search_host_timeseries(fdas_plan_t *p, const void *timeseries_host, float threshold,
                                           fdas_peak_t *peaks_host, int capacity, int *count_host, void *stream)
{
    return search_host_common(p, timeseries_host, true, threshold, peaks_host, capacity, count_host, stream);
}

// Survey form of the host path: series i+1 crosses PCIe while series i is searched.
//   copy stream:    [wait search(i-1)] H2D spectrum(i+1)
//   back stream:    [wait search(i)] D2H count(i), peaks(i)
//   caller stream:  [wait H2D(i)] [wait D2H(i-2)] fdas_search(i)
static int search_host_pipeline(fdas_plan_t *p, const void *spectra_host, bool timeseries, int n_series, float threshold,
                                fdas_peak_t *peaks_host, int capacity, int *counts_host, void *stream)
{
    if (!p || !spectra_host || !counts_host || n_series < 1 || capacity < 0 || (capacity > 0 && !peaks_host))
        return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    const bool plane_free = search_is_plane_free(p);
    int rc = ensure_staging(p, !plane_free, 0);
    if (rc) return rc;
    const size_t spec_bytes = (size_t)p->M * (p->precision == FDAS_F64 ? 16 : 8);
    const size_t in_bytes = timeseries ? (size_t)p->N * sizeof(float) : spec_bytes;   // what crosses the host link per series
    if (timeseries) {
        rc = ensure_staging(p, false, 0);   // stage_spectrum: fdas_spectrum's output, consumed by the search that follows it
        if (rc) return rc;
    }
    rc = ensure_pipe(p);
    if (rc) return rc;
    for (int b = 0; b < 2; ++b) {
        if (!timeseries && !p->pipe_spec[b]) FDAS_CUDA_TRY(p, cudaMalloc(&p->pipe_spec[b], spec_bytes));
        if (timeseries && !p->pipe_series[b]) FDAS_CUDA_TRY(p, cudaMalloc(&p->pipe_series[b], in_bytes));
        if (!p->pipe_count[b]) FDAS_CUDA_TRY(p, cudaMalloc((void **)&p->pipe_count[b], sizeof(int)));
        if (capacity > p->pipe_capacity || !p->pipe_peaks[b]) {
            cudaFree(p->pipe_peaks[b]);
            p->pipe_peaks[b] = NULL;
            FDAS_CUDA_TRY(p, cudaMalloc((void **)&p->pipe_peaks[b], sizeof(fdas_peak_t) * (size_t)(capacity > 0 ? capacity : 1)));
        }
    }
    p->pipe_capacity = capacity;
    cudaStream_t cs = p->pipe_stream, bs = p->pipe_stream_back;
    const unsigned char *src = static_cast<const unsigned char *>(spectra_host);
    void *const *in_buf = timeseries ? p->pipe_series : p->pipe_spec;
    // the pipeline starts after whatever the caller queued on `stream` before this call
    FDAS_CUDA_TRY(p, cudaEventRecord(p->pipe_ev[1][1], st));
    FDAS_CUDA_TRY(p, cudaStreamWaitEvent(cs, p->pipe_ev[1][1], 0));
    FDAS_CUDA_TRY(p, cudaMemcpyAsync(in_buf[0], src, in_bytes, cudaMemcpyHostToDevice, cs));
    FDAS_CUDA_TRY(p, cudaEventRecord(p->pipe_ev[0][0], cs));
    for (int i = 0; i < n_series; ++i) {
        const int b = i & 1;
        FDAS_CUDA_TRY(p, cudaStreamWaitEvent(st, p->pipe_ev[0][b], 0));              // spectrum i is on the device
        if (i >= 2) FDAS_CUDA_TRY(p, cudaStreamWaitEvent(st, p->pipe_ev[2][b], 0));  // peak buffers b were read back
        const void *spec = in_buf[b];
        if (timeseries) {   // the real FFT of PAPER.md:85 on the device, into the one spectrum buffer (stream order protects it)
            rc = fdas_launch_spectrum(p, in_buf[b], p->stage_spectrum, st);
            if (rc) return rc;
            spec = p->stage_spectrum;
        }
        rc = search_on_device(p, spec, plane_free ? NULL : p->stage_plane, threshold, p->pipe_peaks[b], capacity,
                              p->pipe_count[b], st);
        if (rc) return rc;
        FDAS_CUDA_TRY(p, cudaEventRecord(p->pipe_ev[1][b], st));
        if (i + 1 < n_series) {
            // spectrum buffer b^1 was last read by search(i-1), already recorded in pipe_ev[1][b^1]
            if (i >= 1) FDAS_CUDA_TRY(p, cudaStreamWaitEvent(cs, p->pipe_ev[1][b ^ 1], 0));
            FDAS_CUDA_TRY(p, cudaMemcpyAsync(in_buf[b ^ 1], src + (size_t)(i + 1) * in_bytes, in_bytes,
                                             cudaMemcpyHostToDevice, cs));
            FDAS_CUDA_TRY(p, cudaEventRecord(p->pipe_ev[0][b ^ 1], cs));
        }
        // results of series i go back on a stream of their own: the link is full duplex, and behind the copies of the
        // next spectra they would cost every series ~20 us of link time
        FDAS_CUDA_TRY(p, cudaStreamWaitEvent(bs, p->pipe_ev[1][b], 0));
        FDAS_CUDA_TRY(p, cudaMemcpyAsync(counts_host + i, p->pipe_count[b], sizeof(int), cudaMemcpyDeviceToHost, bs));
        if (capacity > 0)
            FDAS_CUDA_TRY(p, cudaMemcpyAsync(peaks_host + (size_t)i * capacity, p->pipe_peaks[b],
                                             sizeof(fdas_peak_t) * (size_t)capacity, cudaMemcpyDeviceToHost, bs));
        FDAS_CUDA_TRY(p, cudaEventRecord(p->pipe_ev[2][b], bs));
    }
    FDAS_CUDA_TRY(p, cudaStreamSynchronize(cs));
    FDAS_CUDA_TRY(p, cudaStreamSynchronize(bs));
    FDAS_CUDA_TRY(p, cudaStreamSynchronize(st));
    return FDAS_OK;
}

extern "C" int fdas_search_host_batched(fdas_plan_t *p, const void *spectra_host, int n_series, float threshold,
                                        fdas_peak_t *peaks_host, int capacity, int *counts_host, void *stream)
{
    return search_host_pipeline(p, spectra_host, false, n_series, threshold, peaks_host, capacity, counts_host, stream);
}

extern "C" int fdas_search_host_timeseries_batched(fdas_plan_t *p, const void *timeseries_host, int n_series, float threshold,
                                                   fdas_peak_t *peaks_host, int capacity, int *counts_host, void *stream)
{
    return search_host_pipeline(p, timeseries_host, true, n_series, threshold, peaks_host, capacity, counts_host, stream);
}

extern "C" int fdas_templates_host(const fdas_plan_t *p, void *dst_host, size_t bytes)
{
    if (!p || !dst_host) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    if (bytes != p->bank_bytes) return FDAS_ERR_INVALID_ARG;
    fdas_plan *q = const_cast<fdas_plan *>(p);
    std::vector<unsigned char> tmp;
    try {
        tmp.resize(bytes);
    } catch (...) {
        return FDAS_ERR_ALLOC;
    }
    FDAS_CUDA_TRY(q, cudaDeviceSynchronize());
    FDAS_CUDA_TRY(q, cudaMemcpy(tmp.data(), p->bank, bytes, cudaMemcpyDeviceToHost));
    // kernel-native order -> natural [K][S]
    const size_t cb = 2 * fdas_storage_scalar_bytes(p->precision);
    const int VC = fdas_bank_vc(p->precision);
    unsigned char *dst = (unsigned char *)dst_host;
    for (int k = 0; k < p->K; ++k)
        for (int f = 0; f < p->S; ++f)
            memcpy(dst + ((size_t)k * p->S + f) * cb, tmp.data() + fdas_bank_offset(k, f, p->T, VC) * cb, cb);
    return FDAS_OK;
}

extern "C" int fdas_taps_host(const fdas_plan_t *p, void *dst_host, size_t bytes)
{
    if (!p || !dst_host) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    if (bytes != (size_t)p->K * (2 * p->m_max + 1) * sizeof(double2)) return FDAS_ERR_INVALID_ARG;
    fdas_plan *q = const_cast<fdas_plan *>(p);
    FDAS_CUDA_TRY(q, cudaDeviceSynchronize());
    FDAS_CUDA_TRY(q, cudaMemcpy(dst_host, p->taps, bytes, cudaMemcpyDeviceToHost));
    return FDAS_OK;
}

extern "C" int fdas_tapmatrix_host(const fdas_plan_t *p, void *dst_host, size_t bytes)
{
    if (!p || !dst_host) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    if (!(p->precision == FDAS_BF16 && p->tc_supported)) return FDAS_ERR_UNSUPPORTED;
    const int ntap = 2 * p->m_max + 1;
    if (bytes != (size_t)p->K * ntap * 2 * sizeof(uint16_t)) return FDAS_ERR_INVALID_ARG;
    fdas_plan *q = const_cast<fdas_plan *>(p);
    const size_t n_tab = (size_t)p->tc_groups * p->tc_nzg;
    std::vector<uint16_t> img;
    std::vector<int2> tab;
    try {
        img.resize(p->tc_bmat_bytes / 2);
        tab.resize(n_tab);
    } catch (...) {
        return FDAS_ERR_ALLOC;
    }
    FDAS_CUDA_TRY(q, cudaDeviceSynchronize());
    FDAS_CUDA_TRY(q, cudaMemcpy(img.data(), p->tc_bmat, p->tc_bmat_bytes, cudaMemcpyDeviceToHost));
    FDAS_CUDA_TRY(q, cudaMemcpy(tab.data(), p->tc_ktab, n_tab * sizeof(int2), cudaMemcpyDeviceToHost));
    // image [g][q][n][e] (kappa = 8 q + e, j = m_max - kappa; column n of (zi, re | im): fdas_tc_column_of_entry)
    // -> natural [K][2 m_max + 1][re, im] with the conjugate for the -|z| rows
    uint16_t *dst = (uint16_t *)dst_host;
    for (int g = 0; g < p->tc_groups; ++g)
        for (int zi = 0; zi < p->tc_nzg; ++zi) {
            const int2 kk = tab[(size_t)g * p->tc_nzg + zi];
            for (int j = -p->m_max; j <= p->m_max; ++j) {
                const int kappa = p->m_max - j;
                const size_t chunk = ((size_t)g * 2 * p->tc_KS + kappa / 8) * p->tc_NT;
                const uint16_t re = img[(chunk + fdas_tc_column_of_entry(zi, 0)) * 8 + kappa % 8];
                const uint16_t im = img[(chunk + fdas_tc_column_of_entry(zi, 1)) * 8 + kappa % 8];
                if (kk.x >= 0) {
                    dst[((size_t)kk.x * ntap + (j + p->m_max)) * 2 + 0] = re;
                    dst[((size_t)kk.x * ntap + (j + p->m_max)) * 2 + 1] = im;
                }
                if (kk.y >= 0 && kk.y != kk.x) {
                    dst[((size_t)kk.y * ntap + (j + p->m_max)) * 2 + 0] = re;
                    dst[((size_t)kk.y * ntap + (j + p->m_max)) * 2 + 1] = (uint16_t)(im ^ 0x8000u);
                }
            }
        }
    return FDAS_OK;
}

extern "C" int fdas_describe_convolve(fdas_plan_t *p, const void *plane_dev, int batch, fdas_kernel_info_t *out)
{
    if (!p || !out || batch < 1) return FDAS_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    if (!plane_dev) return fdas_tc_describe_noplane(p, batch, out);
    if (fdas_uses_mma(p)) {
        const int rc = fdas_tc_describe(p, plane_dev, batch, out);
        // fp32 under FDAS_ALGO_AUTO: a plane buffer the split-operand kernel cannot take goes to the FFT kernel
        if (!(rc == FDAS_ERR_UNSUPPORTED && p->precision == FDAS_F32 && p->algo == FDAS_ALGO_AUTO)) return rc;
    }
    return fdas_fft_describe(p, batch, out);
}

extern "C" int fdas_launch_count(const fdas_plan_t *p, int64_t *count)
{
    if (!p || !count) return FDAS_ERR_INVALID_ARG;
    *count = p->launches;
    return FDAS_OK;
}

extern "C" const char *fdas_status_string(int status)
{
    switch (status) {
    case FDAS_OK: return "FDAS_OK";
    case FDAS_ERR_INVALID_ARG: return "FDAS_ERR_INVALID_ARG";
    case FDAS_ERR_ALLOC: return "FDAS_ERR_ALLOC";
    case FDAS_ERR_CUDA: return "FDAS_ERR_CUDA";
    case FDAS_ERR_NOT_BUILT: return "FDAS_ERR_NOT_BUILT";
    case FDAS_ERR_UNSUPPORTED: return "FDAS_ERR_UNSUPPORTED";
    case FDAS_ERR_TOO_LARGE: return "FDAS_ERR_TOO_LARGE";
    default: return "FDAS_ERR_UNKNOWN";
    }
}

extern "C" int fdas_last_cuda_error(const fdas_plan_t *p)
{
    return p ? (int)p->last_err : -1;
}
