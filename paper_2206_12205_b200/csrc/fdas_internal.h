// fdas_internal.h -- plan layout and helpers shared by the libfdas translation units.
// Product code: never includes or links anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fdas.h"

// Points of the length-S transforms held per thread, and the derived kernel geometry
// (DESIGN.md section 5):  S = 16 * 16 * R3,  T = S/16 threads per segment.
#define FDAS_PTS 16
#define FDAS_MAX_BANDS 32     // harmonic bands one fdas_band_max call can take
#define FDAS_TC_MAX_BOXES 8   // distinct plane-row run lengths the tensor-core kernel's box stores can serve
#define FDAS_TC_MAX_KS 32     // K steps of 16 taps: 2 m_max + 1 <= 512 taps
#define FDAS_TC_STEP_TABLES 9 // K-step tables of the tensor-core kernels: template groups 0..7, then one for every other group

// Kernels that need the opt-in to more than 48 KB of dynamic shared memory.  The opt-in is a per-device function
// attribute; a plan lives on one device, so the largest size requested so far is remembered per plan.
enum {
    FDAS_OPTIN_FFT = 0, FDAS_OPTIN_FFT_SEARCH, FDAS_OPTIN_MMA_BULK, FDAS_OPTIN_MMA_BULK16, FDAS_OPTIN_MMA_SPLIT, FDAS_OPTIN_MMA_SCALAR,
    FDAS_OPTIN_MMA_SCALAR16, FDAS_OPTIN_MMA_NOPLANE, FDAS_OPTIN_MMA_NOPLANE_SPLIT, FDAS_OPTIN_MMA_RECHECK,
    FDAS_OPTIN_MMA_RECHECK_SPLIT, FDAS_OPTIN_RFFT_COLS, FDAS_OPTIN_RFFT_ROWS, FDAS_OPTIN_RFFT_ROWS64, FDAS_OPTIN_HSUM, FDAS_OPTIN_SLOTS
};

struct fdas_plan {
    // problem shape
    int64_t N, M;
    double zmax, dz;
    double jerk;       // w of this slab of the f-fdot-fddot volume (0: plain FDAS)
    int K, S, m_max, L, V, precision;
    int64_t n_seg;
    int T, R3;
    // device objects owned by the plan
    void *bank;        // [K][16/VC][T][VC] complex of the storage type (kernel-native order)
    size_t bank_bytes;
    double2 *taps;     // [K][2*m_max+1] fp64 taps h_z[j], zero padded
    void *twiddle;     // [S] complex of the compute type: exp(+2 pi i j / S)
    int built;
    // tensor-core path of the bf16 variant (fdas_mma.cu): tap matrix image and |z| tables
    int algo;          // fdas_algorithm_t requested by the caller
    int tc_supported;  // the MMA kernel can run this shape
    int tc_groups, tc_nzg, tc_NT, tc_KS, tc_full_chunks;
    unsigned long long tc_nks_lo[8], tc_nks_hi[8];   // columns per K step (nibble = columns / 16; 0 = all), per group
    int tc_ks_first[8];                               // a K step that runs at full width (initialises the accumulators)
    unsigned long long tc_steps[FDAS_TC_STEP_TABLES][FDAS_TC_MAX_KS];   // the K steps in issue order (tc_step_entry, fdas_mma_kernels.cuh)
    int tc_nsteps[FDAS_TC_STEP_TABLES];   // entries of tc_steps[g]
    double tc_cost[8];                    // estimated tensor-pipe cycles per 128-bin tile, per template group
    int tc_rows[8];                       // plane rows of each template group
    int tc_force_scalar_stores;   // testing: run the generic (scalar-store) tensor-core kernel
    void *tc_bmat;     // [groups][2 KS][NT][8] bf16
    size_t tc_bmat_bytes;
    int2 *tc_ktab;     // [groups][nzg] plane rows of (+|z|, -|z|), -1 where absent
    int2 *tc_kref;     // [groups][nzg] (template whose taps fill the columns, its sign)
    int4 *tc_ranges;   // [groups][4] plane-row runs of the bulk kernel's staging rows (row0_n, cnt_n, row0_p, cnt_p;
                       // each cnt carries the index of its tensor-map box in bits 16+)
    int tc_box_heights[FDAS_TC_MAX_BOXES], tc_n_boxes;   // distinct run lengths = box heights of the tensor maps
    int tc_bulk_ok;    // those runs are contiguous (always, for the grids fdas_plan_create builds)
    void *tc_maps;     // host: cached tensor maps of the last plane buffer (fdas_mma.cu)
    const void *tc_maps_plane;
    int tc_maps_batch, tc_maps_elem;
    // NEXT-1: the plane is stored as bf16 bit patterns (fdas_set_plane_format)
    int plane_bf16;
    // fused search (fdas_search): coarse candidates flagged by the convolve epilogue
    fdas_peak_t *cand;     // [cand_capacity] (z_index = first |z| table entry of the chunk, r, chunk maximum)
    int *cand_ctr;         // two counters used alternately: call n appends to [n & 1] and clears [(n + 1) & 1]
    int cand_capacity;
    unsigned search_calls;
    // plane-free search: tile flags / list / counters, the recheck scratch and its tensor maps
    int *tf_flags, *tf_list, *tf_ctr;
    long long tf_tiles;            // entries allocated in tf_flags / tf_list
    float *tf_scratch;
    size_t tf_scratch_bytes;
    void *tf_maps;                 // host: tensor maps of tf_scratch
    unsigned tf_calls;
    // host-buffer entry points: lazily allocated device staging
    void *stage_spectrum, *stage_plane, *stage_series;
    fdas_peak_t *stage_peaks;
    int *stage_count;
    int stage_peaks_capacity;
    void *host_tail;               // pinned host: [count | pad to 16 B | FDAS_TAIL_PEAKS records], the first records of a host search's result
    // fdas_search_host_batched: copy stream, events and double-buffered staging of the host pipeline
    cudaStream_t pipe_stream;
    cudaStream_t pipe_stream_back; // device -> host results of the pipelined host search (the host link is full duplex)
    cudaEvent_t pipe_ev[3][2];     // [h2d done | search done | d2h done][buffer]
    cudaEvent_t chunk_ev[6];       // fdas_search_host: [0] the caller's stream at entry, [1 + c] chunk c of the spectrum on the device
    void *pipe_spec[2], *pipe_series[2];
    fdas_peak_t *pipe_peaks[2];
    int *pipe_count[2];
    int pipe_capacity, pipe_ready;
    // fdas_spectrum: two half-length complex work arrays of the four-step FFT
    void *rfft_scratch;
    // fdas_band_max: per-block partial maxima
    void *band_scratch;
    size_t band_scratch_bytes;
    // bookkeeping
    size_t smem_optin[FDAS_OPTIN_SLOTS];   // dynamic shared memory already opted in to, per kernel kind (this plan's device)
    int device, num_sms;
    cudaError_t last_err;
    int64_t launches;
};

static inline size_t fdas_storage_scalar_bytes(int precision)
{
    return precision == FDAS_F64 ? 8 : (precision == FDAS_F32 ? 4 : 2);
}

static inline size_t fdas_plane_elem_bytes(const fdas_plan *p)
{
    return p->precision == FDAS_F64 ? 8 : (p->plane_bf16 ? 2 : 4);
}

// complexes of the storage type per 16-byte vector: 1 (fp64), 2 (fp32), 4 (bf16)
static inline int fdas_bank_vc(int precision)
{
    return (int)(16 / (2 * fdas_storage_scalar_bytes(precision)));
}

// offset (in complex elements) of H_k[f] inside the kernel-native bank:
// thread t = f % T holds slot a = f / T; slots are grouped VC at a time so that one
// warp-wide 128-bit load covers 512 contiguous bytes.
__host__ __device__ static inline size_t fdas_bank_offset(int k, int f, int T, int VC)
{
    int t = f % T, a = f / T;
    return (((size_t)k * (FDAS_PTS / VC) + a / VC) * T + t) * VC + a % VC;
}

// Column order of the tensor-core tap matrix (fdas_mma.cu): entry pair p = n/4 holds
// (hre_2p, hre_2p+1, him_2p, him_2p+1).
__host__ __device__ static inline int fdas_tc_entry_of_column(int n) { return 2 * (n >> 2) + (n & 1); }
__host__ __device__ static inline int fdas_tc_column_is_imag(int n) { return (n >> 1) & 1; }
__host__ __device__ static inline int fdas_tc_column_of_entry(int zi, int imag) { return 4 * (zi >> 1) + (zi & 1) + 2 * imag; }

// What the convolve epilogue needs to flag candidates for fdas_search (enabled = 0: plain convolve).
struct fdas_search_args {
    int enabled;
    float thr;
    fdas_peak_t *cand;
    int *cand_count;       // appended to by this launch
    int *cand_count_next;  // cleared by this launch for the next call
    int cand_capacity;
    int *count_out;        // caller's peak counter, cleared by this launch
    int cand_span;         // |z| table entries one candidate covers (set by the convolve launch)
    // plane-free search (fdas_search with plane_dev == NULL; fdas_mma_search.cu): the scan launch flags the 128-bin
    // tiles that hold a cell above the threshold, the recheck launch recomputes those tiles and applies the peak rule
    int *tile_flags;       // [batch * tiles_per_series]: bit 0 = a cell above thr; bits 1, 2 = its first / last bin is one
    int *tile_list;        // flagged tiles (series * tiles_per_series + tile), each appended once
    int *tile_count;       // entries of tile_list: this call's counter ...
    int *tile_count_next;  // ... and the other one, cleared by the scan launch for the next call
    float *scratch;        // recheck launch: [gridDim.x][K][FDAS_TC_STRIP] powers of the tiles of one work item
    fdas_peak_t *peaks;    // [batch][capacity] records out
    int capacity;
    int *counts;           // [batch] totals out (cleared by the scan launch)
};
#define FDAS_TAIL_PEAKS 1024    // records fetched together with the count by the host search forms (one synchronisation)
#define FDAS_TC_STRIP 384   // bins per recheck work item: the flagged tile and its two neighbours

#define FDAS_CUDA_TRY(p, call)                                  \
    do {                                                        \
        cudaError_t e__ = (call);                               \
        if (e__ != cudaSuccess) {                               \
            if (p) (p)->last_err = e__;                         \
            return FDAS_ERR_CUDA;                               \
        }                                                       \
    } while (0)

template <class Kern>
static inline int fdas_optin_smem(fdas_plan *p, int slot, Kern kern, size_t bytes)
{
    if (bytes <= p->smem_optin[slot] || bytes <= 48u * 1024u) return FDAS_OK;
    FDAS_CUDA_TRY(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    p->smem_optin[slot] = bytes;
    return FDAS_OK;
}

// implemented in fdas_templates.cu / fdas_convolve.cu / fdas_peaks.cu
int fdas_launch_build_templates(fdas_plan *p, cudaStream_t st);
int fdas_launch_convolve(fdas_plan *p, const void *spectra, void *planes, int batch, cudaStream_t st);
// fdas_mma.cu: host-side grouping (plan creation), tap matrix build, the tcgen05 convolution
int fdas_mma_plan(fdas_plan *p);
int fdas_launch_build_tapmatrix(fdas_plan *p, cudaStream_t st);
int fdas_launch_convolve_mma(fdas_plan *p, const void *spectra, void *planes, int batch, cudaStream_t st,
                             fdas_search_args *search = nullptr);
// fdas_mma_search.cu: convolve + peaks without a plane (scan launch + recheck launch); FDAS_ERR_UNSUPPORTED when
// the plan does not run the tensor-core kernels with a float plane format
int fdas_launch_search_noplane(fdas_plan *p, const void *spectra, int batch, float thr, fdas_peak_t *peaks, int capacity,
                               int *counts, cudaStream_t st);
// the same in steps (fdas_mma_search.cu): begin, scan launches over block ranges, one recheck launch
int fdas_launch_resolve3(fdas_plan *p, const void *volume, int n_slabs, int slab, const fdas_search_args &sa, fdas_peak3_t *peaks,
                         int capacity, int *count, cudaStream_t st);
int fdas_launch_convolve_fft_search(fdas_plan *p, const void *spectrum, void *plane, const fdas_search_args *search, cudaStream_t st);
int fdas_launch_resolve_cells(fdas_plan *p, const void *plane, const fdas_search_args &sa, fdas_peak_t *peaks, int capacity, cudaStream_t st);
int fdas_search_prepare(fdas_plan *p, float thr, int *count_dev, cudaStream_t st, fdas_search_args *sa);   // fdas_plan.cu
int fdas_noplane_block_bins(const fdas_plan *p, int batch);
int fdas_noplane_begin(fdas_plan *p, int batch, float thr, fdas_peak_t *peaks, int capacity, int *counts, cudaStream_t st,
                       fdas_search_args *out);
int fdas_noplane_scan(fdas_plan *p, const void *spectra, int batch, const fdas_search_args *sa, int blk_first, int n_blk,
                      cudaStream_t st);
int fdas_noplane_recheck(fdas_plan *p, const void *spectra, int batch, const fdas_search_args *sa, cudaStream_t st);
// fdas_mma.cu: the work-item size the tensor-core launch picks, and tensor maps of a [rows][cols] matrix with one box
// per distinct run length (shared with fdas_mma_search.cu)
int fdas_tc_encode_maps(fdas_plan *p, void *base, long long cols, long long rows, size_t elem_bytes, void *maps_out);
// what fdas_convolve_batched would launch (fdas_describe_convolve): tensor-core forms (fdas_mma.cu; the scan launch of the
// plane-free search when plane_dev is NULL, fdas_mma_search.cu) and the overlap-save FFT form (fdas_convolve.cu)
int fdas_tc_describe(fdas_plan *p, const void *plane_dev, int batch, fdas_kernel_info_t *out);
int fdas_tc_describe_noplane(fdas_plan *p, int batch, fdas_kernel_info_t *out);
int fdas_fft_describe(fdas_plan *p, int batch, fdas_kernel_info_t *out);
double fdas_tc_issued_flops(const fdas_plan *p, int batch, int plane_free);
int fdas_tc_trims(const fdas_plan *p, bool plane_free);   // does this launch skip the columns a K step does not reach?
// fdas_peaks.cu: turns the candidates of a fused search into the peak list (same rule as fdas_peaks)
int fdas_launch_resolve(fdas_plan *p, const void *plane, const fdas_search_args &sa, fdas_peak_t *peaks, int capacity,
                        cudaStream_t st);
// true when fdas_convolve runs the tensor-core kernel for this plan
static inline int fdas_uses_mma(const fdas_plan *p)
{
    if (!p->tc_supported || p->algo == FDAS_ALGO_FFT) return 0;
    if (p->precision == FDAS_BF16) return 1;
    // fp32 variant: split-operand form (bf16 x 3), box stores only -> 16-byte aligned plane rows
    return p->precision == FDAS_F32 && p->M % 4 == 0 && !p->tc_force_scalar_stores;
}
int fdas_launch_peaks(fdas_plan *p, const void *plane, float thr, fdas_peak_t *peaks, int capacity,
                      int *count, cudaStream_t st);
// fdas_peaks.cu: 26-neighbour peak rule over a volume of n_slabs planes of this plan's shape
int fdas_launch_peaks3(fdas_plan *p, const void *volume, int n_slabs, float thr, fdas_peak3_t *peaks, int capacity, int *count,
                       cudaStream_t st);
// fdas_harmonic.cu: S_H[k][r] = sum_h P[k0 + h (k - k0)][h r]
int fdas_launch_harmonic_sum(fdas_plan *p, const void *plane, void *sum, int n_harmonics, int k0, int drift, cudaStream_t st);
// fdas_rfft.cu: the real FFT ahead of the convolution
int fdas_launch_spectrum(fdas_plan *p, const void *timeseries, void *spectrum, cudaStream_t st);
// fdas_bands.cu: Table 3 band maxima
int fdas_launch_band_max(fdas_plan *p, const void *plane, double f_bin, int n_bands, fdas_peak_t *out, cudaStream_t st);
// fdas_cast.cu: the paper's quick cast of a bf16-stored plane
int fdas_launch_quick_cast(fdas_plan *p, const void *src_bf16, void *dst_f32, long long n, cudaStream_t st);
