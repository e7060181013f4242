// fdas_volume.cu -- the f-fdot-fddot volume of a jerk search (include/fdas.h: fdas_volume_*).
//
// PAPER.md:71-73 (section 2.2): "Jerk Searching takes into account a change in acceleration, and therefore extends
// the f-fdot plane into an f-fdot-fddot volume.  More candidate templates are required to populate the third
// dimension ... based on the same principal of convolving templates."  A volume is a stack of slabs, one per jerk
// value w_i = -wmax + i dw (the grid rule of z); slab i is an ordinary plan whose K templates all carry the jerk
// w_i (fdas_plan_create_jerk, reading A25), so every slab runs the convolution kernels of the plain
// search -- tensor-core form or overlap-save FFT form -- on the SAME spectrum in device memory.  Peaks are taken
// over the volume: the plane rule with one more axis (26 neighbours, reading A27).
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "fdas_internal.h"

struct fdas_volume {
    int n_slabs;
    double wmax, dw;
    fdas_plan **slabs;
    int built;
    // host-buffer entry point: one spectrum staging shared by all slabs, the volume, the peak list
    void *stage_spectrum, *stage_volume;
    fdas_peak3_t *stage_peaks;
    int *stage_count;
    int stage_peaks_capacity;
    cudaError_t last_err;
    int64_t launches;   // launches of the volume's own kernels (the slabs count theirs)
};

#define FDAS_VOL_TRY(v, call)                                   \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) {                               \
            (v)->last_err = e__;                                \
            return FDAS_ERR_CUDA;                               \
        }                                                       \
    } while (0)

extern "C" int fdas_volume_destroy(fdas_volume_t *v)
{
    if (!v) return FDAS_OK;
    if (v->slabs)
        for (int i = 0; i < v->n_slabs; ++i) fdas_plan_destroy(v->slabs[i]);   // synchronises the device
    free(v->slabs);
    cudaFree(v->stage_spectrum);
    cudaFree(v->stage_volume);
    cudaFree(v->stage_peaks);
    cudaFree(v->stage_count);
    delete v;
    return FDAS_OK;
}

extern "C" int fdas_volume_create(fdas_volume_t **out, int64_t N, double zmax, double dz, double wmax, double dw, int seglen,
                                  int precision)
{
    if (!out) return FDAS_ERR_INVALID_ARG;
    *out = NULL;
    if (!(wmax >= 0.0) || !(dw > 0.0) || !isfinite(wmax) || !isfinite(dw)) return FDAS_ERR_INVALID_ARG;
    const double nn = floor(wmax / dw + 1e-9);
    if (nn > 255.0) return FDAS_ERR_INVALID_ARG;
    fdas_volume *v = new (std::nothrow) fdas_volume;
    if (!v) return FDAS_ERR_ALLOC;
    memset(v, 0, sizeof(*v));
    v->n_slabs = 2 * (int)nn + 1;
    v->wmax = wmax;
    v->dw = dw;
    v->slabs = (fdas_plan **)calloc((size_t)v->n_slabs, sizeof(fdas_plan *));
    if (!v->slabs) {
        delete v;
        return FDAS_ERR_ALLOC;
    }
    for (int i = 0; i < v->n_slabs; ++i) {
        const int rc = fdas_plan_create_jerk(&v->slabs[i], N, zmax, dz, -wmax + i * dw, seglen, precision);
        if (rc != FDAS_OK) {   // the widest slab (|w| = wmax) decides whether the segment length is enough
            fdas_volume_destroy(v);
            return rc;
        }
    }
    *out = v;
    return FDAS_OK;
}

extern "C" int fdas_volume_info(const fdas_volume_t *v, fdas_volume_info_t *info)
{
    if (!v || !info) return FDAS_ERR_INVALID_ARG;
    const fdas_plan *p = v->slabs[0];
    info->n_slabs = v->n_slabs;
    info->n_templates = p->K;
    info->n_bins = p->M;
    info->precision = p->precision;
    info->elem_bytes = fdas_plane_elem_bytes(p);
    info->wmax = v->wmax;
    info->dw = v->dw;
    return FDAS_OK;
}

extern "C" int fdas_volume_w_of_index(const fdas_volume_t *v, int i, double *w)
{
    if (!v || !w || i < 0 || i >= v->n_slabs) return FDAS_ERR_INVALID_ARG;
    *w = -v->wmax + i * v->dw;
    return FDAS_OK;
}

extern "C" int fdas_volume_slab(const fdas_volume_t *v, int i, fdas_plan_t **plan)
{
    if (!v || !plan || i < 0 || i >= v->n_slabs) return FDAS_ERR_INVALID_ARG;
    *plan = v->slabs[i];
    return FDAS_OK;
}

extern "C" int fdas_volume_set_algorithm(fdas_volume_t *v, int algorithm)
{
    if (!v) return FDAS_ERR_INVALID_ARG;
    for (int i = 0; i < v->n_slabs; ++i) {
        const int rc = fdas_set_algorithm(v->slabs[i], algorithm);
        if (rc) return rc;
    }
    return FDAS_OK;
}

extern "C" int fdas_volume_build_templates(fdas_volume_t *v, void *stream)
{
    if (!v) return FDAS_ERR_INVALID_ARG;
    for (int i = 0; i < v->n_slabs; ++i) {
        const int rc = fdas_build_templates(v->slabs[i], stream);
        if (rc) return rc;
    }
    v->built = 1;
    return FDAS_OK;
}

extern "C" int fdas_volume_convolve(fdas_volume_t *v, const void *spectrum_dev, void *volume_dev, void *stream)
{
    if (!v || !spectrum_dev || !volume_dev) return FDAS_ERR_INVALID_ARG;
    if (!v->built) return FDAS_ERR_NOT_BUILT;
    const fdas_plan *p0 = v->slabs[0];
    const size_t slab_bytes = (size_t)p0->K * p0->M * fdas_plane_elem_bytes(p0);
    for (int i = 0; i < v->n_slabs; ++i) {
        const int rc = fdas_convolve(v->slabs[i], spectrum_dev, static_cast<unsigned char *>(volume_dev) + (size_t)i * slab_bytes, stream);
        if (rc) {
            v->last_err = v->slabs[i]->last_err;
            return rc;
        }
    }
    return FDAS_OK;
}

extern "C" int fdas_volume_peaks(fdas_volume_t *v, const void *volume_dev, float threshold, fdas_peak3_t *peaks_dev, int capacity,
                                 int *count_dev, void *stream)
{
    if (!v || !volume_dev || !count_dev || capacity < 0 || (capacity > 0 && !peaks_dev)) return FDAS_ERR_INVALID_ARG;
    fdas_plan *p0 = v->slabs[0];
    const int rc = fdas_launch_peaks3(p0, volume_dev, v->n_slabs, threshold, peaks_dev, capacity, count_dev, (cudaStream_t)stream);
    if (rc) v->last_err = p0->last_err;
    else v->launches += 1;
    return rc;
}

extern "C" int fdas_volume_search(fdas_volume_t *v, const void *spectrum_dev, void *volume_dev, float threshold,
                                  fdas_peak3_t *peaks_dev, int capacity, int *count_dev, void *stream)
{
    if (!v || !spectrum_dev || !volume_dev || !count_dev || capacity < 0 || (capacity > 0 && !peaks_dev)) return FDAS_ERR_INVALID_ARG;
    if (!v->built) return FDAS_ERR_NOT_BUILT;
    // Tensor-core slabs with a float volume: every slab's convolve launch flags its candidate cells (the fused threshold
    // of fdas_search), then one small launch per slab applies the 26-neighbour rule to those cells only -- the volume
    // (8 GB for 5 slabs of config 3) is not read back.  Other plans: convolve, then the full peak pass.
    bool fused = true;
    for (int i = 0; i < v->n_slabs; ++i) fused = fused && fdas_uses_mma(v->slabs[i]) && !v->slabs[i]->plane_bf16;
    if (fused) {
        cudaStream_t st = (cudaStream_t)stream;
        const fdas_plan *p0 = v->slabs[0];
        const size_t slab_elems = (size_t)p0->K * p0->M;
        fdas_search_args *sa = new (std::nothrow) fdas_search_args[v->n_slabs];
        if (!sa) return FDAS_ERR_ALLOC;
        int rc = FDAS_OK;
        for (int i = 0; i < v->n_slabs && rc == FDAS_OK; ++i) {
            rc = fdas_search_prepare(v->slabs[i], threshold, count_dev, st, &sa[i]);
            if (rc == FDAS_OK)
                rc = fdas_launch_convolve_mma(v->slabs[i], spectrum_dev, static_cast<float *>(volume_dev) + (size_t)i * slab_elems, 1, st, &sa[i]);
            if (rc == FDAS_ERR_UNSUPPORTED && i == 0) {   // this volume buffer cannot take the box stores (alignment): plain path
                v->slabs[0]->search_calls -= 1;
                fused = false;
                rc = FDAS_OK;
                break;
            }
        }
        if (fused) {
            // every convolve launch cleared count_dev; the resolve launches add to it
            for (int i = 0; i < v->n_slabs && rc == FDAS_OK; ++i)
                rc = fdas_launch_resolve3(v->slabs[i], volume_dev, v->n_slabs, i, sa[i], peaks_dev, capacity, count_dev, st);
            delete[] sa;
            return rc;
        }
        delete[] sa;
    }
    const int rc = fdas_volume_convolve(v, spectrum_dev, volume_dev, stream);
    if (rc) return rc;
    return fdas_volume_peaks(v, volume_dev, threshold, peaks_dev, capacity, count_dev, stream);
}

extern "C" int fdas_volume_search_host(fdas_volume_t *v, const void *spectrum_host, float threshold, fdas_peak3_t *peaks_host,
                                       int capacity, int *count_host, void *stream)
{
    if (!v || !spectrum_host || !count_host || capacity < 0 || (capacity > 0 && !peaks_host)) return FDAS_ERR_INVALID_ARG;
    if (!v->built) return FDAS_ERR_NOT_BUILT;
    cudaStream_t st = (cudaStream_t)stream;
    const fdas_plan *p0 = v->slabs[0];
    const size_t spec_bytes = (size_t)p0->M * (p0->precision == FDAS_F64 ? 16 : 8);
    const size_t vol_bytes = (size_t)v->n_slabs * p0->K * p0->M * fdas_plane_elem_bytes(p0);
    if (!v->stage_spectrum) FDAS_VOL_TRY(v, cudaMalloc(&v->stage_spectrum, spec_bytes));
    if (!v->stage_volume) FDAS_VOL_TRY(v, cudaMalloc(&v->stage_volume, vol_bytes));
    if (!v->stage_count) FDAS_VOL_TRY(v, cudaMalloc((void **)&v->stage_count, sizeof(int)));
    if (capacity > v->stage_peaks_capacity) {
        cudaFree(v->stage_peaks);
        v->stage_peaks = NULL;
        v->stage_peaks_capacity = 0;
        FDAS_VOL_TRY(v, cudaMalloc((void **)&v->stage_peaks, sizeof(fdas_peak3_t) * (size_t)capacity));
        v->stage_peaks_capacity = capacity;
    }
    // the spectrum crosses the host link ONCE and feeds every slab
    FDAS_VOL_TRY(v, cudaMemcpyAsync(v->stage_spectrum, spectrum_host, spec_bytes, cudaMemcpyHostToDevice, st));
    const int rc = fdas_volume_search(v, v->stage_spectrum, v->stage_volume, threshold, v->stage_peaks, capacity, v->stage_count, stream);
    if (rc) return rc;
    FDAS_VOL_TRY(v, cudaMemcpyAsync(count_host, v->stage_count, sizeof(int), cudaMemcpyDeviceToHost, st));
    FDAS_VOL_TRY(v, cudaStreamSynchronize(st));
    const int n = *count_host < capacity ? *count_host : capacity;
    if (n > 0) {
        FDAS_VOL_TRY(v, cudaMemcpyAsync(peaks_host, v->stage_peaks, sizeof(fdas_peak3_t) * (size_t)n, cudaMemcpyDeviceToHost, st));
        FDAS_VOL_TRY(v, cudaStreamSynchronize(st));
    }
    return FDAS_OK;
}

extern "C" int fdas_volume_launch_count(const fdas_volume_t *v, int64_t *count)
{
    if (!v || !count) return FDAS_ERR_INVALID_ARG;
    int64_t n = v->launches;
    for (int i = 0; i < v->n_slabs; ++i) n += v->slabs[i]->launches;
    *count = n;
    return FDAS_OK;
}

extern "C" int fdas_volume_last_cuda_error(const fdas_volume_t *v)
{
    return v ? (int)v->last_err : -1;
}
