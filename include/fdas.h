/*
 * fdas.h -- C ABI of libfdas: the FDAS (Fourier Domain Acceleration Search) Fourier-domain
 * convolution stage of arxiv 2206.12205 ("Bits missing: Finding exotic pulsars using
 * bfloat16 on NVIDIA GPUs"), written from scratch for NVIDIA B200 (sm_100a).
 *
 * PAPER.md below is /root/reference/PAPER.md (text of the paper); DESIGN.md is this repo's.
 *
 * What the library computes:
 *   the complex spectrum X[0..M-1] of a time series is convolved with a bank of K
 *   constant-acceleration response templates h_z (Ransom et al. 2002, cited PAPER.md:37)
 *   by the overlap-save method (Fig. 1), and the squared magnitude is
 *   written as the f-fdot power plane
 *        P[k][r] = | sum_{j=-m_k..m_k} X[r-j] h_{z_k}[j] |^2 ,  k = 0..K-1, r = 0..M-1,
 *   with X = 0 outside [0, M), z_k = -zmax + k*dz, m_k = ceil(|z_k|/2) + 16, and
 *   h_z[j] = conj( int_0^1 exp(2 pi i [ j u + (z/2)(u^2 - u) ]) du ).
 *   Three precisions: fp64 ("gold standard"), fp32, and bf16 storage with
 *   fp32 accumulation.
 *
 * Conventions
 *   - Every function returns an fdas_status_t as int (0 = FDAS_OK).  The library never
 *     throws, exits or prints.
 *   - All pointers named *_dev are DEVICE pointers (e.g. a torch tensor's data_ptr()),
 *     16-byte aligned.  Pointers named *_host are HOST pointers.  The caller owns them.
 *     The library owns the plan and everything inside it (template bank, twiddle tables).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All
 *     GPU work is enqueued on it.  Only the *_host entry points and fdas_plan_destroy
 *     synchronise.
 *   - Output is bit-reproducible run to run (no atomics touch the plane).  The ORDER of
 *     peak records is unspecified.
 *   - A plan may be used from one host thread and on one stream at a time (its scratch buffers, candidate
 *     lists and tensor-map caches are per plan, not per call); distinct plans are independent.  A plan
 *     belongs to the device that was current when it was created; that device must be current in every call.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns
 *     FDAS_ERR_CUDA.
 */
#ifndef FDAS_H_
#define FDAS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FDAS_VERSION_MAJOR 0
#define FDAS_VERSION_MINOR 1

typedef struct fdas_plan fdas_plan_t; /* opaque */

/* Arithmetic / storage variant. */
typedef enum {
    FDAS_F64 = 0,  /* complex128 spectrum, fp64 bank and FFTs, double plane              */
    FDAS_F32 = 1,  /* complex64 spectrum, fp32 templates, fp32 accumulation, float plane; see
                      fdas_set_algorithm for the two evaluation orders                     */
    FDAS_BF16 = 2  /* complex64 spectrum rounded to bf16 on load (RNE), bf16 templates, fp32
                      accumulation, float plane ("bf16 storage / fp32 accumulate"; DESIGN.md
                      reading A12); see fdas_set_algorithm for the two evaluation orders     */
} fdas_precision_t;

/* How fdas_convolve evaluates the convolution (fdas_set_algorithm). */
typedef enum {
    FDAS_ALGO_AUTO = 0, /* default: FDAS_ALGO_MMA where it applies (FDAS_BF16; FDAS_F32 with M % 4 == 0),
                           else FDAS_ALGO_FFT                                                  */
    FDAS_ALGO_FFT = 1,  /* overlap-save FFTs on the fp32/fp64 ALUs, all precisions */
    FDAS_ALGO_MMA = 2,  /* FDAS_BF16 and FDAS_F32: the same linear convolution as a tensor-core
                           contraction over the taps (tcgen05, bf16 operands, fp32 accumulation), no
                           FFT.  FDAS_F32 splits every fp32 operand into two bf16 terms            */
    FDAS_ALGO_MMA_SCALAR = 3 /* FDAS_ALGO_MMA with the plane written by per-thread stores instead of
                           shared-memory staging + bulk copies: the form FDAS_ALGO_MMA falls back
                           to when M % 4 != 0.  Same arithmetic, bit-identical plane; selectable
                           so that tests and profiles can compare the two store paths.      */
} fdas_algorithm_t;

/* Element type of the power plane written by fdas_convolve (fdas_set_plane_format). */
typedef enum {
    FDAS_PLANE_F32 = 0, /* default: float (double in FDAS_F64)                                   */
    FDAS_PLANE_BF16 = 1 /* bfloat16 bit patterns (uint16): the paper's bfloat16 pipeline keeps the
                           f-fdot plane in bfloat16 and widens it afterwards by the "quick cast"
                           (PAPER.md:91-93); halves the dominant HBM stream of the path        */
} fdas_plane_format_t;

typedef enum {
    FDAS_OK = 0,
    FDAS_ERR_INVALID_ARG = 1, /* NULL pointer, bad size, illegal parameter combination   */
    FDAS_ERR_ALLOC = 2,       /* host or device allocation failed                        */
    FDAS_ERR_CUDA = 3,        /* a CUDA call failed; see fdas_last_cuda_error            */
    FDAS_ERR_NOT_BUILT = 4,   /* convolve/peaks before fdas_build_templates              */
    FDAS_ERR_UNSUPPORTED = 5, /* legal request this build has no kernel for              */
    FDAS_ERR_TOO_LARGE = 6    /* beyond the fixed capacity of a call that allocates nothing (fdas_search_static) */
} fdas_status_t;

/* One peak candidate (12 bytes). */
typedef struct {
    int32_t z_index; /* k, row of the plane; z = -zmax + k*dz                            */
    int32_t r;       /* Fourier bin                                                      */
    float power;     /* P[k][r] (rounded to float in FDAS_F64 mode)                      */
} fdas_peak_t;

typedef struct {
    int64_t n_bins;          /* M = N/2 spectrum bins = plane columns                    */
    int32_t n_templates;     /* K = 2*floor(zmax/dz) + 1                                 */
    int32_t seglen;          /* S, overlap-save segment FFT length                       */
    int32_t halfwidth_max;   /* m_max = ceil(zmax/2) + 16                                */
    int32_t overlap_left;    /* L >= m_max: segment s starts at bin s*V - L              */
    int32_t valid_per_seg;   /* V <= S - L - m_max: bins written per segment             */
    int32_t precision;       /* fdas_precision_t                                         */
    int64_t n_segments;      /* ceil(M / V)                                              */
    int64_t plane_row_pitch; /* elements between plane rows (= M: rows are contiguous)   */
    size_t plane_elem_bytes; /* 4 (float), 8 (double, FDAS_F64) or 2 (FDAS_PLANE_BF16)           */
    size_t spectrum_elem_bytes; /* 8 (complex64) or 16 (complex128, FDAS_F64)            */
    size_t bank_bytes;       /* device bytes of the template bank                        */
} fdas_info_t;

/*
 * fdas_plan_create -- fix the problem shape (BASELINE.json north_star: "fdas_plan_create(N,
 * zmax, dz, seglen, precision)").
 *   N        real samples of the time series; the spectrum has M = N/2 bins (bins
 *            0..N/2-1 of the real FFT, Nyquist dropped; reading A8).  N even,
 *            N >= 2*seglen.
 *   zmax,dz  template grid z_k = -zmax + k*dz (Eq. 1: z = Fourier bin
 *            drift).  zmax >= 0, dz > 0, K <= 4096.
 *   seglen   overlap-save FFT length S: one of 256, 512, 1024, 2048,
 *            4096, and S - 2*m_max >= 32.
 *   precision fdas_precision_t.
 * Allocates the template bank and tables on the current CUDA device.  *out is set to NULL
 * on failure.  Errors: INVALID_ARG, UNSUPPORTED (seglen 8192), ALLOC, CUDA.
 */
int fdas_plan_create(fdas_plan_t **out, int64_t N, double zmax, double dz, int seglen,
                     int precision);

/*
 * fdas_plan_create_jerk -- one slab of the f-fdot-fddot volume of a jerk search (PAPER.md:71-73,
 * section 2.2: "Jerk Searching takes into account a change in acceleration, and therefore extends
 * the f-fdot plane into an f-fdot-fddot volume.  More candidate templates are required to populate
 * the third dimension ... based on the same principal of convolving templates").  The plan is an
 * ordinary FDAS plan whose K templates all carry the jerk `w` (change of the drift z over the
 * observation, in Fourier bins; reading A25):
 *      h_{z,w}[j] = conj( int_0^1 exp(2 pi i [ j u + (z/2)(u^2 - u) + (w/12)(2u^3 - 3u^2 + u) ]) du ),
 *      |j| <= m = ceil(|z|/2 + |w|/12) + 16,
 * i.e. the response of a signal of mean frequency r0 and mean drift z whose frequency follows
 * r0 + z (u - 1/2) + (w/2)(u^2 - u + 1/6).  A volume is a set of such plans, one per w; every other
 * entry point (convolve, search, peaks, harmonic sum, ...) acts on one slab.  The +-z pairing that the
 * tensor-core form uses survives the jerk (h_{-z,w} = conj h_{z,w}); the taps are no longer even in j.
 * w = 0 is fdas_plan_create.  Same errors; seglen must leave S - L - m >= 32 with the wider taps.
 */
int fdas_plan_create_jerk(fdas_plan_t **out, int64_t N, double zmax, double dz, double w, int seglen,
                          int precision);

/*
 * fdas_set_algorithm -- choose how fdas_convolve evaluates Y_z[r] = sum_j X[r-j] h_z[j]
 * (PAPER.md:35, :59).  Both algorithms compute the same plane; they differ in rounding points:
 *   FDAS_ALGO_FFT  overlap-save FFTs; in FDAS_BF16 the spectrum, the FFT'd
 *                  bank and every inter-pass exchange are rounded to bf16.
 *   FDAS_ALGO_MMA  FDAS_BF16: the spectrum and the taps h_z[j] are rounded to bf16 once (RNE) and
 *                  the sum over the <= 2 m_max + 1 taps runs on the tensor cores with fp32
 *                  accumulation ("bf16 storage / fp32 accumulate", north_star).  Needs
 *                  m_max <= 255.
 *                  FDAS_F32: spectrum and fp32 taps are each split exactly into bf16 terms,
 *                  x = x1 + x2 + r with x1 = bf16(x), x2 = bf16(x - x1), |r| <= 2^-17 |x|, and the
 *                  three leading products x1 h1 + x1 h2 + x2 h1 are accumulated in fp32; the
 *                  dropped terms are <= 2^-17 of each product, an order of magnitude inside the
 *                  fp32 tolerance (|dP| <= 1e-4 P_peak + 1e-4; measured 3e-6 P_peak).  Needs
 *                  M % 4 == 0 (16-byte aligned plane rows); other sizes run FDAS_ALGO_FFT.
 * Errors: INVALID_ARG (NULL, unknown value), UNSUPPORTED (FDAS_ALGO_MMA on an FDAS_F64 plan, on
 * an FDAS_F32 plan with M % 4 != 0, or on a plan whose taps do not fit; FDAS_ALGO_MMA_SCALAR on
 * anything but FDAS_BF16).  fdas_get_algorithm reports the algorithm fdas_convolve
 * will run (FDAS_ALGO_FFT, FDAS_ALGO_MMA or FDAS_ALGO_MMA_SCALAR, never AUTO).
 */
int fdas_set_algorithm(fdas_plan_t *p, int algorithm);
int fdas_get_algorithm(const fdas_plan_t *p, int *algorithm);

/*
 * fdas_set_plane_format -- choose the element type of the plane (section 3.1).
 *   FDAS_PLANE_BF16  FDAS_BF16 plans on the tensor-core algorithm only.  Every power is computed
 *                    in fp32 exactly as for FDAS_PLANE_F32 and rounded once, to nearest even, to
 *                    bfloat16; plane_dev of fdas_convolve / fdas_convolve_batched / fdas_search /
 *                    fdas_peaks and plane_host of fdas_convolve_host are then [K][M] uint16 bit
 *                    patterns (fdas_info_t.plane_elem_bytes = 2).  fdas_peaks and fdas_search
 *                    apply the peak rule to the stored (rounded) values; rounding creates ties,
 *                    which the rule's ordering resolves (one peak per plateau).
 * Errors: INVALID_ARG (NULL, unknown value), UNSUPPORTED (bf16 plane on a plan that does not run
 * the tensor-core kernels; fdas_set_algorithm(FDAS_ALGO_FFT) while the plane format is bf16).
 */
int fdas_set_plane_format(fdas_plan_t *p, int format);
int fdas_get_plane_format(const fdas_plan_t *p, int *format);

/*
 * fdas_quick_cast -- the paper's widening of a bf16-stored plane ("copying the two
 * bytes of data for each bfloat16 number into the corresponding positions of an all zero
 * single-precision output array").  plane_bf16_dev: batch*K*M uint16; plane_f32_dev: batch*K*M
 * float, fully overwritten: word i = (uint32) bits[i] << 16, bit-exact.  The two buffers must not
 * overlap.  Works for any plan (only K and M are used).  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, batch < 1), CUDA.
 */
int fdas_quick_cast(fdas_plan_t *p, const void *plane_bf16_dev, void *plane_f32_dev, int batch, void *stream);

/*
 * fdas_harmonic_sum -- gather the power of the harmonics of every cell ("diminishing
 * harmonics at integer multiples of both f and fdot.  The summed height (power) of the peak and
 * harmonics is typically used to calculate the signal-to-noise ratio").  Plain
 * definition (reading A23):
 *      S[k][r] = sum_{h=1..n_harmonics} P[k0 + h (k - k0)][h r],    k0 = (K-1)/2, the row of z = 0,
 * terms whose row or bin falls outside the plane are skipped.
 *   plane_dev  [K][M] in the plan's plane format (float, double for FDAS_F64, bf16 bits)
 *   sum_dev    [K][M] float (double for FDAS_F64), fully overwritten; must not overlap plane_dev
 *   n_harmonics 1..32 (1 copies / widens the plane)
 * The result is a plane like any other: fdas_peaks accepts it when the plan's plane format is
 * float.  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, n_harmonics out of range), UNSUPPORTED (z = 0 is not a row of the
 * template grid, i.e. zmax is not a multiple of dz: harmonics would fall between rows), CUDA.
 */
int fdas_harmonic_sum(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, void *stream);

/*
 * fdas_harmonic_sum_drift -- the drift-tolerant form ("Quantisation error in both the
 * frequency and acceleration axes of the search lead to the observed peaks drifting into adjacent
 * bins.  To account for this, a harmonic sum algorithm is used").  DESIGN.md reading A26: a signal
 * detected in cell (k, r) lies within half a cell of it, so its h-th harmonic lies within h/2 cells of
 * (k0 + h (k - k0), h r); harmonic h contributes the LARGEST power of that window:
 *      S'[k][r] = sum_h max_{|dk|,|dr| <= floor(h/2)} P[k0 + h (k - k0) + dk][h r + dr]
 * (window cells outside the plane are skipped; S' >= S of fdas_harmonic_sum; n_harmonics = 1 gives
 * the plane).  Arguments, types and errors as fdas_harmonic_sum.
 */
int fdas_harmonic_sum_drift(fdas_plan_t *p, const void *plane_dev, void *sum_dev, int n_harmonics, void *stream);

/*
 * fdas_band_max -- the paper's own peak selection (section 4.3, Table 3): the
 * plane is split into harmonic bands derived from the fundamental frequency f and "the n-th
 * harmonic is taken to be the highest point in the n-th band".  Band 0 (fundamental) holds the
 * bins 0 <= r <= 1.5 f, band n >= 1 the bins (n + 0.5) f < r <= (n + 1.5) f (upper bound
 * inclusive, Table 3's caption), over all K rows.
 *   plane_dev  [K][M] in the plan's plane format
 *   f_bin      fundamental frequency in Fourier bins (f T), > 0
 *   n_bands    1..32
 *   out_dev    n_bands records (z_index, r, power); among equal maxima the first in (k, r) order;
 *              (-1, -1, 0) for a band that lies beyond the plane
 * Asynchronous on `stream`; scratch memory is owned by the plan (allocated on first use).
 * Errors: INVALID_ARG, CUDA.
 */
int fdas_band_max(fdas_plan_t *p, const void *plane_dev, double f_bin, int n_bands, fdas_peak_t *out_dev, void *stream);

/* Frees the plan and its device memory (synchronises the device first).  NULL is OK. */
int fdas_plan_destroy(fdas_plan_t *p);

/* Copies the derived sizes into *info. */
int fdas_plan_info(const fdas_plan_t *p, fdas_info_t *info);

/* z_k = -zmax + k*dz for 0 <= k < K. */
int fdas_z_of_index(const fdas_plan_t *p, int k, double *z);

/*
 * fdas_build_templates -- the template builder ("Each template is a 1D array
 * of complex numbers ... generated ... then ... converted to bfloat16/double-precision by a
 * tuned GPU kernel"; response function PAPER.md:37).  A GPU kernel evaluates the taps
 * h_z[j], j = -m_z..m_z, in fp64, a second one takes their length-S DFT with the 1/S of the
 * inverse transform folded in, H_z[f] = (1/S) sum_j h_z[j] exp(-2 pi i f j / S), and rounds
 * once to the bank's storage type (fp64 / fp32 / bf16 RNE; reading A11).
 * Asynchronous on `stream`.  Must complete (stream order) before fdas_convolve.
 */
int fdas_build_templates(fdas_plan_t *p, void *stream);

/*
 * fdas_spectrum -- the "Real FFT" that feeds the convolution (Fig. 1; :85 "intentionally
 * left in single-precision"): X[k] = (1/sqrt N) sum_j x[j] exp(-2 pi i j k / N), k = 0..N/2-1
 * (Nyquist dropped; unit-variance noise gives unit mean power per bin, readings A8, A9).
 *   timeseries_dev  N floats (the plan's N), 16-byte aligned
 *   spectrum_dev    M = N/2 interleaved complex in the plan's spectrum type (float2; double2 for
 *                   FDAS_F64, widened from the fp32 result as in the paper's pipeline)
 * fp32 arithmetic throughout.  N must be a power of two, 2^10 <= N <= 2^23.  Work arrays (8 N bytes)
 * are owned by the plan and allocated on first use.  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL), UNSUPPORTED (N not a power of two in range), ALLOC, CUDA.
 */
int fdas_spectrum(fdas_plan_t *p, const void *timeseries_dev, void *spectrum_dev, void *stream);

/*
 * fdas_convolve -- the fused hot path (PAPER.md:65-67 overlap-save; :59 power plane).
 * One kernel: per segment, load S bins (zero outside [0,M)), forward FFT once, then for
 * every template multiply by H_z, inverse FFT, |.|^2, and store only the V valid bins.
 *   spectrum_dev  M interleaved complex (float2 for F32/BF16, double2 for F64)
 *   plane_dev     [K][M] row-major, float (F32/BF16) or double (F64); fully overwritten
 * Asynchronous on `stream`; no host synchronisation.
 * Errors: INVALID_ARG (NULL), NOT_BUILT, CUDA.
 */
int fdas_convolve(fdas_plan_t *p, const void *spectrum_dev, void *plane_dev, void *stream);

/*
 * Batched form for independent series sharing one bank (BASELINE.json config 4):
 * spectra_dev [batch][M], planes_dev [batch][K][M], both contiguous.  batch >= 1.
 */
int fdas_convolve_batched(fdas_plan_t *p, const void *spectra_dev, void *planes_dev, int batch,
                          void *stream);

/*
 * fdas_peaks -- threshold / local-maximum pass over one plane (the
 * analysis takes "the highest point" of a band; reading A14).  (k, r) is reported
 * iff P[k][r] > threshold and P[k][r] >= each of its (up to 8) existing neighbours, strictly
 * greater than those that precede it in (k, r) lexicographic order.
 *   peaks_dev   device array of `capacity` records (may be NULL iff capacity == 0)
 *   count_dev   device int32: receives the TOTAL number of peaks found (snprintf
 *               convention: only min(count, capacity) records are written; overflow is not
 *               an error).  The call zeroes it first, on `stream`.
 * Record order is unspecified.  Asynchronous on `stream`.
 */
int fdas_peaks(fdas_plan_t *p, const void *plane_dev, float threshold, fdas_peak_t *peaks_dev,
               int capacity, int *count_dev, void *stream);

/*
 * fdas_search -- fdas_convolve followed by fdas_peaks in one call: the same plane in plane_dev
 * and the same peak set.  Where the convolution runs on the tensor-core
 * path the threshold test is fused into its epilogue: the kernel flags the (rare) cells above
 * `threshold` while it stores them and a small second kernel applies the local-maximum rule to
 * those cells only, so the plane is never read back from HBM.  Other plans run the two kernels
 * of fdas_convolve and fdas_peaks.  Arguments, ownership and the snprintf convention for
 * count_dev are those of fdas_convolve and fdas_peaks.  Asynchronous on `stream`.
 *
 * plane_dev == NULL: the PLANE-FREE form (what a search keeps of the plane is its peak
 * list; surveys run batches of 256 series whose planes nobody reads).  Nothing but the
 * spectrum is read from HBM and nothing but the peak list is written: a first launch runs the whole
 * convolution without storing, listing the 128-bin tiles that hold a power above `threshold`; a second launch
 * recomputes the listed tiles (the same tensor-core instructions and the same fp32 arithmetic, so every power is
 * bit-identical to what fdas_convolve stores) and applies the peak rule there.  The peak set and the powers equal
 * those of the call with a plane.  Cost grows with the number of listed tiles: with a threshold inside the
 * noise every tile is listed and the call costs about four convolutions.  Needs a plan that runs the
 * tensor-core kernels (fdas_get_algorithm != FDAS_ALGO_FFT; FDAS_F32 with M % 4 == 0) with the float plane
 * format and at most 8 template groups (K <= 1023 on a symmetric grid); otherwise FDAS_ERR_UNSUPPORTED.
 */
int fdas_search(fdas_plan_t *p, const void *spectrum_dev, void *plane_dev, float threshold,
                fdas_peak_t *peaks_dev, int capacity, int *count_dev, void *stream);

/*
 * fdas_search_static -- the plane-free fdas_search (plane_dev == NULL) of one series for callers that cannot
 * allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The call makes NO
 * cudaMalloc / cudaFree and calls no allocating library routine: the scratch the two launches share (tile flags, tile
 * list, two counters) lives in a device array compiled into the library, 262 400 bytes that every GPU loading the
 * library holds until the process exits.  Same kernels and arithmetic as fdas_search: the same peak set, the same
 * power bits.  The caller passes inputs and outputs as for fdas_search.
 *   limit      M = N/2 <= FDAS_SEARCH_STATIC_MAX_BINS (2^22 bins, BASELINE.json config 3), one series per call, one
 *              template group (K <= 127 on a symmetric grid: configs 1-4)
 *   sharing    every call, of every plan and stream, uses the same array, which keeps the last call's contents: the
 *              call clears what must start at zero (stream-ordered, before its first launch), and two calls that
 *              overlap on the GPU (different streams, no ordering between them) RACE -- order them
 *   device     the plan's device must be current (the array's address is looked up per device, once)
 *   capture    a plan's first call sets function attributes and looks the address up: make it before a stream capture;
 *              later calls consist of one memset and two kernel launches and can be captured into a CUDA graph
 * Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, capacity < 0, another device current), NOT_BUILT, TOO_LARGE (M beyond the limit),
 * UNSUPPORTED (a plan the plane-free fdas_search does not take, or more than one template group), CUDA.
 */
#define FDAS_SEARCH_STATIC_MAX_BINS 4194304
int fdas_search_static(fdas_plan_t *p, const void *spectrum_dev, float threshold, fdas_peak_t *peaks_dev,
                       int capacity, int *count_dev, void *stream);

/*
 * fdas_search_batched -- fdas_search over `batch` independent series sharing the plan (BASELINE.json config 4).
 *   spectra_dev  [batch][M]
 *   planes_dev   [batch][K][M], or NULL for the plane-free form: ONE scan launch and ONE recheck launch
 *                for the whole batch (config 4's 256 planes would be 208 GB)
 *   peaks_dev    [batch][capacity] records; series b's first min(counts_dev[b], capacity) are valid
 *   counts_dev   [batch] totals (snprintf convention per series)
 * Per series the peak set equals that of fdas_search.  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, batch < 1, capacity < 0), NOT_BUILT, UNSUPPORTED (plane-free form, see fdas_search), ALLOC, CUDA.
 */
int fdas_search_batched(fdas_plan_t *p, const void *spectra_dev, void *planes_dev, int batch, float threshold,
                        fdas_peak_t *peaks_dev, int capacity, int *counts_dev, void *stream);

/*
 * Host-buffer forms (end-to-end path): copy the spectrum host->device, run fdas_convolve
 * (and fdas_peaks), copy the result device->host, on `stream`, then synchronise the stream.
 * Device staging buffers are owned by the plan and allocated on first use.  Pinned host
 * memory makes the copies asynchronous and fast; pageable memory also works.
 *   fdas_convolve_host   plane_host receives [K][M]
 *   fdas_search_host     fdas_search in its plane-free form where the plan allows it (no plane is allocated
 *                        anywhere), else with a plane that stays on the device; peaks_host
 *                        receives min(count, capacity) records and *count_host the total.  In the plane-free
 *                        form a spectrum of 8 MB or more is copied in five chunks (1/2, 1/4, 1/8, 1/16, 1/16) on a stream of the plan's own
 *                        (ordered after `stream` at entry) and every chunk is scanned as soon as the next one
 *                        has landed, so the search overlaps the copy; the result is the same.
 */
int fdas_convolve_host(fdas_plan_t *p, const void *spectrum_host, void *plane_host, void *stream);
int fdas_search_host(fdas_plan_t *p, const void *spectrum_host, float threshold,
                     fdas_peak_t *peaks_host, int capacity, int *count_host, void *stream);

/*
 * fdas_search_host_batched -- survey form of fdas_search_host for many independent series sharing
 * one plan (BASELINE.json config 4; PAPER.md:295-297 times 256-run batches): series i+1 is copied
 * host->device on an internal copy stream while series i is searched on `stream` (plane-free where the plan
 * allows it; otherwise one device plane buffer is reused); only the peak lists come back.
 *   spectra_host  [n_series][M] interleaved complex (pinned memory makes the overlap real)
 *   peaks_host    [n_series][capacity] records; for series i the first min(counts_host[i], capacity)
 *                 are valid (the whole slot of `capacity` records is copied: keep capacity modest)
 *   counts_host   [n_series] total number of peaks found per series (snprintf convention)
 * Per series the peak SET equals that of fdas_search_host.  Synchronises `stream` before returning.
 * Errors: INVALID_ARG (NULL, n_series < 1, capacity < 0), NOT_BUILT, ALLOC, CUDA.
 */
int fdas_search_host_batched(fdas_plan_t *p, const void *spectra_host, int n_series, float threshold,
                             fdas_peak_t *peaks_host, int capacity, int *counts_host, void *stream);

/*
 * fdas_search_host_timeseries / _batched -- the end-to-end flow of the paper's Fig. 1 from the TIME SERIES
 * (PAPER.md:63-67, :85): the N fp32 samples are copied host->device (the same bytes as the spectrum they replace),
 * fdas_spectrum takes the real FFT on the device, fdas_search follows.  timeseries_host: [N] floats
 * ([n_series][N] for the batched form, whose copy of series i+1 overlaps the FFT and search of series i).
 * Every other argument, the result and the errors are those of fdas_search_host / fdas_search_host_batched, plus
 * fdas_spectrum's UNSUPPORTED (N not a power of two in 2^10 .. 2^23).
 */
int fdas_search_host_timeseries(fdas_plan_t *p, const void *timeseries_host, float threshold,
                                fdas_peak_t *peaks_host, int capacity, int *count_host, void *stream);
int fdas_search_host_timeseries_batched(fdas_plan_t *p, const void *timeseries_host, int n_series, float threshold,
                                        fdas_peak_t *peaks_host, int capacity, int *counts_host, void *stream);

/*
 * Debug / test access to the bank: copies H_z[f] in NATURAL order, [K][S] interleaved
 * complex of the storage type (double2 / float2 / 2 x bf16 bit patterns), to host memory.
 * `bytes` must equal K*S*2*sizeof(storage scalar).  Synchronises.
 * fdas_taps_host copies the fp64 taps: for template k, 2*m_max+1 complex doubles
 * (zero-padded beyond m_k), j = -m_max..m_max.  `bytes` = K*(2*m_max+1)*16.
 */
int fdas_templates_host(const fdas_plan_t *p, void *dst_host, size_t bytes);
int fdas_taps_host(const fdas_plan_t *p, void *dst_host, size_t bytes);
/*
 * FDAS_BF16 plans only: the bf16 taps the tensor-core path multiplies with (PAPER.md:105
 * "converted to bfloat16"), un-permuted from its tap-matrix image: [K][2*m_max+1][2] uint16
 * bit patterns (re, im), j = -m_max..m_max.  `bytes` = K*(2*m_max+1)*4.  Synchronises.
 * Errors: UNSUPPORTED when the plan has no tap matrix.
 */
int fdas_tapmatrix_host(const fdas_plan_t *p, void *dst_host, size_t bytes);

/*
 * ---- f-fdot-fddot volume: the jerk search (section 2.2: "extends the f-fdot plane into an f-fdot-fddot
 * volume.  More candidate templates are required to populate the third dimension") ------------------------------------
 * A volume is a stack of slabs V[i][k][r], one per jerk value w_i = -wmax + i*dw, i = 0..2*floor(wmax/dw) (the grid
 * rule of z; w = change of the drift z over the observation, in Fourier bins); slab i is the plane of
 * fdas_plan_create_jerk(.., w_i, ..) (reading A25).  The volume object owns one plan per slab; all slabs are
 * convolved from the same spectrum in device memory.
 *   fdas_volume_create          same arguments and errors as fdas_plan_create_jerk, plus the w grid (wmax >= 0, dw > 0,
 *                               at most 511 slabs); the segment length must fit the widest taps (|w| = wmax)
 *   fdas_volume_slab            the plan of slab i (borrowed: do not destroy it), e.g. for fdas_set_plane_format
 *   fdas_volume_set_algorithm   fdas_set_algorithm on every slab
 *   fdas_volume_build_templates fdas_build_templates on every slab (asynchronous on `stream`)
 *   fdas_volume_convolve        volume_dev [n_slabs][K][M] in the slabs' plane format, fully overwritten
 *   fdas_volume_peaks           (i, k, r) is reported iff V > threshold and V >= each of its (up to 26) existing
 *                               neighbours, strictly greater than those that precede it in (i, k, r) lexicographic
 *                               order: the rule of fdas_peaks with one more axis (reading A27; a plateau
 *                               yields one peak).  snprintf convention for count_dev; record order unspecified
 *   fdas_volume_search          fdas_volume_convolve + fdas_volume_peaks
 *   fdas_volume_search_host     host spectrum in (copied to the device ONCE for all slabs), peak list out; the
 *                               volume stays in device memory owned by the volume object; synchronises `stream`
 * Errors as for the plan calls they wrap.
 */
typedef struct fdas_volume fdas_volume_t; /* opaque */
typedef struct {
    int32_t w_index; /* i, slab of the volume; w = -wmax + i*dw                          */
    int32_t z_index; /* k, row of the slab; z = -zmax + k*dz                             */
    int32_t r;       /* Fourier bin                                                      */
    float power;     /* V[i][k][r]                                                       */
} fdas_peak3_t;
typedef struct {
    int32_t n_slabs;     /* W = 2*floor(wmax/dw) + 1                                      */
    int32_t n_templates; /* K rows per slab                                               */
    int64_t n_bins;      /* M                                                             */
    int32_t precision;   /* fdas_precision_t                                              */
    size_t elem_bytes;   /* bytes per volume element (the slabs' plane format)            */
    double wmax, dw;
} fdas_volume_info_t;
int fdas_volume_create(fdas_volume_t **out, int64_t N, double zmax, double dz, double wmax, double dw, int seglen,
                       int precision);
int fdas_volume_destroy(fdas_volume_t *v); /* NULL is OK; synchronises the device */
int fdas_volume_info(const fdas_volume_t *v, fdas_volume_info_t *info);
int fdas_volume_w_of_index(const fdas_volume_t *v, int i, double *w);
int fdas_volume_slab(const fdas_volume_t *v, int i, fdas_plan_t **plan);
int fdas_volume_set_algorithm(fdas_volume_t *v, int algorithm);
int fdas_volume_build_templates(fdas_volume_t *v, void *stream);
int fdas_volume_convolve(fdas_volume_t *v, const void *spectrum_dev, void *volume_dev, void *stream);
int fdas_volume_peaks(fdas_volume_t *v, const void *volume_dev, float threshold, fdas_peak3_t *peaks_dev, int capacity,
                      int *count_dev, void *stream);
int fdas_volume_search(fdas_volume_t *v, const void *spectrum_dev, void *volume_dev, float threshold,
                       fdas_peak3_t *peaks_dev, int capacity, int *count_dev, void *stream);
int fdas_volume_search_host(fdas_volume_t *v, const void *spectrum_host, float threshold, fdas_peak3_t *peaks_host,
                            int capacity, int *count_host, void *stream);
int fdas_volume_launch_count(const fdas_volume_t *v, int64_t *count);
int fdas_volume_last_cuda_error(const fdas_volume_t *v);

/*
 * fdas_describe_convolve -- what fdas_convolve_batched(p, ., plane_dev, batch, .) would launch, so that a benchmark
 * can name the kernel it times and count its work without restating the launcher.  plane_dev is
 * only inspected for its alignment (the tensor-core form stores through tensor maps when the plane rows are 16-byte
 * aligned); plane_dev == NULL describes the scan launch of the plane-free fdas_search.  Launches nothing.
 * Errors: INVALID_ARG, UNSUPPORTED (plane-free form on a plan that cannot run it).
 */
typedef struct {
    int32_t algorithm;         /* FDAS_ALGO_FFT, FDAS_ALGO_MMA or FDAS_ALGO_MMA_SCALAR                               */
    int32_t split;             /* tensor-core forms: 1 = bf16 operands, 3 = fp32 operands as 3 products of bf16 terms;
                                  0 = FFT form                                                                      */
    int32_t groups;            /* template groups (more than one when the bank holds more than 128 templates)       */
    int32_t nch, k_steps;      /* tensor-core forms: UMMA N = 16 nch columns per part, K steps of 16 taps           */
    int32_t work_item_bins;    /* bins per work item (tensor-core forms) / valid bins per segment (FFT form)        */
    int32_t grid_x, grid_y, block_threads;   /* tensor-core forms: a one-dimensional grid, the template groups share
                                                its CTAs in proportion to their work per tile (grid_y = 1)             */
    size_t dynamic_smem_bytes;
    double tensor_flops;       /* dense MMA flops the launch issues, padding included (0 for the FFT form)          */
    char kernel[128];          /* kernel name with its template arguments                                           */
} fdas_kernel_info_t;
int fdas_describe_convolve(fdas_plan_t *p, const void *plane_dev, int batch, fdas_kernel_info_t *out);

/* Number of kernels this plan has launched so far (template build + convolve + peaks). */
int fdas_launch_count(const fdas_plan_t *p, int64_t *count);

const char *fdas_status_string(int status);

/* Last cudaError_t seen by this plan, as int (0 = cudaSuccess).  -1 if p is NULL. */
int fdas_last_cuda_error(const fdas_plan_t *p);

#ifdef __cplusplus
}
#endif
#endif /* FDAS_H_ */
