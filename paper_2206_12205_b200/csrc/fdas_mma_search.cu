// fdas_mma_search.cu -- plane-free search (include/fdas.h: fdas_search / fdas_search_batched with a NULL plane).
//
// PAPER.md:184-188 (section 4.3): what a search keeps of the f-fdot plane is a list of peaks, not the plane;
// PAPER.md:295-297 (section 5.4) times batches of 256 series, whose planes (BASELINE.json config 4: 208 GB) nobody
// reads.  SURVEY.md 8(f) NEXT-2: emit the candidates from the convolution itself and skip the plane write.
//
// Two launches of the tensor-core kernel (fdas_mma_kernels.cuh), no plane in HBM:
//   TB_SCAN     the whole convolution, powers formed in registers exactly as for a plane, nothing stored; every
//               128-bin tile holding a power above the threshold is listed (a few hundred of 32 768 on config 3)
//   TB_RECHECK  the listed tiles (with the neighbour tile where a first / last bin is a candidate) are computed
//               again by the same MMAs and the same epilogue arithmetic -- bit-identical to what fdas_convolve
//               stores -- into a per-CTA strip of scratch memory ([K][384] floats, L2 resident), and the epilogue
//               warps apply the peak rule of fdas_peaks to the cells of the listed tile.
// The peak set (and every power) equals that of fdas_search with a float plane.  The only HBM stream left is the
// spectrum read: the path is bound by the tensor pipe (bf16 operands) instead of the plane write.
#include <stdio.h>
#include <stdlib.h>
#include <mutex>
#include "fdas_mma_kernels.cuh"

namespace {

template <int NCH, int SPLIT, int MODE>
int launch_mode(fdas_plan *p, const TcParams &tp, unsigned gx, size_t smem_bytes, const TbMaps *maps, cudaStream_t st)
{
    auto kern = fdas_mma_bulk_kernel<NCH, float, SPLIT, MODE>;
    const int slot = MODE == TB_SCAN ? (SPLIT == 3 ? FDAS_OPTIN_MMA_NOPLANE_SPLIT : FDAS_OPTIN_MMA_NOPLANE)
                                     : (SPLIT == 3 ? FDAS_OPTIN_MMA_RECHECK_SPLIT : FDAS_OPTIN_MMA_RECHECK);
    { const int rc = fdas_optin_smem(p, slot, kern, smem_bytes); if (rc) return rc; }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = MODE == TB_RECHECK ? dim3(gx, p->tc_groups) : dim3(gx);   // scan: one-dimensional, every group's CTAs (TcParams::cta0)
    cfg.blockDim = dim3(tb_threads(SPLIT));
    cfg.dynamicSmemBytes = smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (MODE == TB_RECHECK && p->tc_groups > 1) {   // the template groups of one work item meet at a cluster barrier
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = 1;
        attr[na].val.clusterDim.y = (unsigned)p->tc_groups;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    if (MODE == TB_RECHECK) {   // programmatic dependent of the scan launch: set up while it drains, griddepcontrol.wait inside
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    FDAS_CUDA_TRY(p, cudaLaunchKernelEx(&cfg, kern, tp, *maps));
    p->launches += 1;
    return FDAS_OK;
}

template <int SPLIT, int MODE>
int launch_nch(fdas_plan *p, const TcParams &tp, unsigned gx, size_t smem_bytes, const TbMaps *maps, cudaStream_t st)
{
    switch (p->tc_NT / 16) {
    case 1: return launch_mode<1, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 2: return launch_mode<2, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 3: return launch_mode<3, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 4: return launch_mode<4, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 5: return launch_mode<5, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 6: return launch_mode<6, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 7: return launch_mode<7, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    case 8: return launch_mode<8, SPLIT, MODE>(p, tp, gx, smem_bytes, maps, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}

}  // namespace

// work item of the scan launch: as for a plane (the largest of 1024..128 bins that fits and leaves two items per CTA)
static int scan_item_bins(const fdas_plan *p, int batch, int split, int sms_per_group)
{
    int R = 1024;
    for (;; R >>= 1) {
        const long long items = (long long)batch * ((p->M + R - 1) / R);
        if (R == 128 || (TbSmem(R, p->tc_KS, p->tc_NT, TC_TILE * 4, split, false).total <= 227u * 1024u && items >= 2LL * sms_per_group)) break;
    }
    return fdas_tc_balance_items(R, p->M, batch, sms_per_group);
}

int fdas_tc_describe_noplane(fdas_plan *p, int batch, fdas_kernel_info_t *out)
{
    if (!fdas_uses_mma(p) || p->plane_bf16 || !p->tc_bulk_ok || p->tc_groups > 8) return FDAS_ERR_UNSUPPORTED;
    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    const int R = scan_item_bins(p, batch, split, sms_per_group);
    const long long items = (long long)batch * ((p->M + R - 1) / R);
    out->algorithm = FDAS_ALGO_MMA;
    out->split = split;
    out->groups = p->tc_groups;
    out->nch = p->tc_NT / 16;
    out->k_steps = p->tc_KS;
    out->work_item_bins = R;
    {
        TcParams tp;
        tc_fill_params(p, tp, nullptr, nullptr, batch, R);
        out->grid_x = (int32_t)fdas_tc_split_ctas(p, tp, items);
        out->grid_y = 1;
    }
    out->block_threads = tb_threads(split);
    out->dynamic_smem_bytes = TbSmem(R, p->tc_KS, p->tc_NT, TC_TILE * 4, split, false).total;
    out->tensor_flops = fdas_tc_issued_flops(p, batch, 1);
    snprintf(out->kernel, sizeof(out->kernel), "fdas_mma_bulk_kernel<%d, float, %d, TB_SCAN> (+ TB_RECHECK on the listed tiles)", p->tc_NT / 16, split);
    return FDAS_OK;
}

// The plane-free search in three steps, so that a caller can scan a series range by range (fdas_search_host scans
// the chunks of the spectrum as they arrive over the host link):
//   fdas_noplane_begin    buffers, counters, the arguments both launches share
//   fdas_noplane_scan     scan launch over blocks [blk_first, blk_first + n_blk) of every series (n_blk <= 0: all);
//                         block = the scan's work item, fdas_noplane_block_bins() bins
//   fdas_noplane_recheck  recheck launch over every tile listed since fdas_noplane_begin
int fdas_noplane_block_bins(const fdas_plan *p, int batch)
{
    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    return scan_item_bins(p, batch, split, sms_per_group);
}

int fdas_noplane_begin(fdas_plan *p, int batch, float thr, fdas_peak_t *peaks, int capacity, int *counts, cudaStream_t st,
                       fdas_search_args *out)
{
    // the tensor-core kernels with a float plane format; the strip stores need the row runs of the box-store path; the
    // template groups of one item must fit one cluster
    if (!fdas_uses_mma(p) || p->plane_bf16 || !p->tc_bulk_ok || p->tc_groups > 8) return FDAS_ERR_UNSUPPORTED;
    const long long tps = (p->M + TC_TILE - 1) / TC_TILE;
    const long long tiles = (long long)batch * tps;
    if (tiles >= 0x7FFFFFFFLL) return FDAS_ERR_UNSUPPORTED;
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;

    // ---- buffers: tile flags (all zero between calls: the recheck launch clears what the scan launch set), tile list,
    // two counters used alternately, the recheck strips and their tensor maps
    if (tiles > p->tf_tiles) {
        cudaFree(p->tf_flags);
        cudaFree(p->tf_list);
        p->tf_flags = p->tf_list = NULL;
        p->tf_tiles = 0;
        int *f = NULL, *l = NULL;
        cudaError_t e = cudaMalloc((void **)&f, sizeof(int) * (size_t)tiles);
        if (e == cudaSuccess) e = cudaMalloc((void **)&l, sizeof(int) * (size_t)tiles);
        if (e == cudaSuccess) e = cudaMemsetAsync(f, 0, sizeof(int) * (size_t)tiles, st);
        if (e != cudaSuccess) {
            cudaFree(f);
            cudaFree(l);
            p->last_err = e;
            return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
        }
        p->tf_flags = f;
        p->tf_list = l;
        p->tf_tiles = tiles;
    }
    if (!p->tf_ctr) {
        FDAS_CUDA_TRY(p, cudaMalloc((void **)&p->tf_ctr, 2 * sizeof(int)));
        FDAS_CUDA_TRY(p, cudaMemsetAsync(p->tf_ctr, 0, 2 * sizeof(int), st));
    }
    const size_t strip_bytes = (size_t)sms_per_group * p->K * FDAS_TC_STRIP * sizeof(float);
    if (!p->tf_scratch) {
        FDAS_CUDA_TRY(p, cudaMalloc(&p->tf_scratch, strip_bytes));
        p->tf_scratch_bytes = strip_bytes;
        if (!p->tf_maps) p->tf_maps = aligned_alloc(64, sizeof(TbMaps));
        if (!p->tf_maps) return FDAS_ERR_ALLOC;
        const int rc = fdas_tc_encode_maps(p, p->tf_scratch, FDAS_TC_STRIP, (long long)sms_per_group * p->K, sizeof(float), p->tf_maps);
        if (rc != FDAS_OK) {
            cudaFree(p->tf_scratch);
            p->tf_scratch = NULL;
            return rc;
        }
    }
    fdas_search_args sa = {};
    sa.enabled = 1;
    sa.thr = thr;
    sa.cand_span = 8;
    sa.tile_flags = p->tf_flags;
    sa.tile_list = p->tf_list;
    sa.tile_count = p->tf_ctr + (p->tf_calls & 1);
    sa.tile_count_next = p->tf_ctr + ((p->tf_calls + 1) & 1);
    sa.scratch = p->tf_scratch;
    sa.peaks = peaks;
    sa.capacity = capacity;
    sa.counts = counts;
    p->tf_calls += 1;
    *out = sa;
    return FDAS_OK;
}

int fdas_noplane_scan(fdas_plan *p, const void *spectra, int batch, const fdas_search_args *sa, int blk_first, int n_blk,
                      cudaStream_t st)
{
    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    const int R = scan_item_bins(p, batch, split, sms_per_group);
    const uint32_t total = TbSmem(R, p->tc_KS, p->tc_NT, TC_TILE * 4, split, false).total;
    if (total > 227u * 1024u) return FDAS_ERR_UNSUPPORTED;
    TcParams tp;
    tc_fill_params(p, tp, spectra, nullptr, batch, R);
    if (n_blk > 0) {
        if (blk_first < 0 || blk_first + n_blk > tp.n_blocks) return FDAS_ERR_INVALID_ARG;
        tp.blk_first = blk_first;
        tp.n_blocks = n_blk;
    }
    tp.search = *sa;
    const long long items = (long long)batch * tp.n_blocks;
    if (items >= 0x7FFFFFFFLL) return FDAS_ERR_UNSUPPORTED;
    const unsigned gx = fdas_tc_split_ctas(p, tp, items);
    const TbMaps *maps = static_cast<const TbMaps *>(p->tf_maps);
    return split == 3 ? launch_nch<3, TB_SCAN>(p, tp, gx, total, maps, st) : launch_nch<1, TB_SCAN>(p, tp, gx, total, maps, st);
}

// one CTA (one cluster of template groups) per strip; CTAs without a listed tile leave at once
int fdas_noplane_recheck(fdas_plan *p, const void *spectra, int batch, const fdas_search_args *sa, cudaStream_t st)
{
    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    const long long tiles = (long long)batch * ((p->M + TC_TILE - 1) / TC_TILE);
    // one template group: the strip of the listed tile sits in shared memory; several: staging rows for the box
    // stores into the scratch strips the groups share
    const uint32_t total = TbSmem(FDAS_TC_STRIP, p->tc_KS, p->tc_NT, TC_TILE * 4, split, true, p->tc_groups == 1 ? p->K : 0).total;
    if (total > 227u * 1024u) return FDAS_ERR_UNSUPPORTED;
    TcParams tp;
    tc_fill_params(p, tp, spectra, nullptr, batch, FDAS_TC_STRIP);
    tp.search = *sa;
    tp.clustered = p->tc_groups > 1;
    const unsigned gx = (unsigned)(tiles < sms_per_group ? tiles : sms_per_group);
    const TbMaps *maps = static_cast<const TbMaps *>(p->tf_maps);
    return split == 3 ? launch_nch<3, TB_RECHECK>(p, tp, gx, total, maps, st) : launch_nch<1, TB_RECHECK>(p, tp, gx, total, maps, st);
}

int fdas_launch_search_noplane(fdas_plan *p, const void *spectra, int batch, float thr, fdas_peak_t *peaks, int capacity,
                               int *counts, cudaStream_t st)
{
    fdas_search_args sa;
    int rc = fdas_noplane_begin(p, batch, thr, peaks, capacity, counts, st, &sa);
    if (rc == FDAS_OK) rc = fdas_noplane_scan(p, spectra, batch, &sa, 0, 0, st);
    if (rc == FDAS_OK) rc = fdas_noplane_recheck(p, spectra, batch, &sa, st);
    return rc;
}

// =====================================================================================
// fdas_search_static (include/fdas.h): the plane-free search of ONE series with every byte of scratch in a
// file-scope device array, for callers that may not allocate (CUDA graph capture, serving loops).  Same two
// launches, same kernels, same arithmetic as fdas_launch_search_noplane; only where the tile flags, the tile list
// and the two counters live differs.  One template group only: the recheck launch then keeps its strip in shared
// memory and needs no scratch strip in global memory (and no tensor map).
// =====================================================================================
#define FDAS_STATIC_TILES (FDAS_SEARCH_STATIC_MAX_BINS / 128)   // 128-bin tiles of the longest series accepted
#define FDAS_STATIC_CTR_INTS 64                                 // the two counters, padded to 256 bytes
// [0, 64): counters | [64, 64 + TILES): tile flags | [64 + TILES, 64 + 2 TILES): tile list.  262 400 bytes, held by
// every GPU that loads the library until the process exits; shared by every call, so calls that overlap on the GPU race.
static __device__ __align__(256) int fdas_static_scratch[FDAS_STATIC_CTR_INTS + 2 * FDAS_STATIC_TILES];

// Device address of the array on the CURRENT device.  In host code `fdas_static_scratch` is a host-side stand-in for
// the symbol, not a device address: the address comes from cudaGetSymbolAddress, once per device, with that device
// current (the caller checks that the plan's device is).
static int static_scratch_address(fdas_plan *p, int **out)
{
    constexpr int MAX_DEV = 64;
    static int *addr[MAX_DEV];
    static std::mutex mu;
    std::lock_guard<std::mutex> lock(mu);
    const int dev = p->device;
    if (dev >= 0 && dev < MAX_DEV && addr[dev]) {
        *out = addr[dev];
        return FDAS_OK;
    }
    int *ptr = nullptr;
    FDAS_CUDA_TRY(p, cudaGetSymbolAddress((void **)&ptr, fdas_static_scratch));
    if (!ptr) return FDAS_ERR_CUDA;
    if (dev >= 0 && dev < MAX_DEV) addr[dev] = ptr;
    *out = ptr;
    return FDAS_OK;
}

extern "C" int fdas_search_static(fdas_plan_t *p, const void *spectrum_dev, float threshold, fdas_peak_t *peaks_dev,
                                  int capacity, int *count_dev, void *stream)
{
    if (!p || !spectrum_dev || !count_dev || capacity < 0 || (capacity > 0 && !peaks_dev)) return FDAS_ERR_INVALID_ARG;
    if (!p->built) return FDAS_ERR_NOT_BUILT;
    // the same plans as the plane-free fdas_search, with one template group
    if (!fdas_uses_mma(p) || p->plane_bf16 || !p->tc_bulk_ok || p->tc_groups != 1) return FDAS_ERR_UNSUPPORTED;
    if (p->M > (long long)FDAS_SEARCH_STATIC_MAX_BINS) return FDAS_ERR_TOO_LARGE;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = -1;
    FDAS_CUDA_TRY(p, cudaGetDevice(&dev));
    if (dev != p->device) return FDAS_ERR_INVALID_ARG;   // the scratch address below is that of the current device
    int *scratch = nullptr;
    { const int rc = static_scratch_address(p, &scratch); if (rc) return rc; }

    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const int tiles = (int)((p->M + TC_TILE - 1) / TC_TILE);
    const int R = scan_item_bins(p, 1, split, p->num_sms);
    const uint32_t scan_smem = TbSmem(R, p->tc_KS, p->tc_NT, TC_TILE * 4, split, false).total;
    const uint32_t recheck_smem = TbSmem(FDAS_TC_STRIP, p->tc_KS, p->tc_NT, TC_TILE * 4, split, true, p->K).total;
    if (scan_smem > 227u * 1024u || recheck_smem > 227u * 1024u) return FDAS_ERR_UNSUPPORTED;

    // the array keeps what the last call (of any plan, on any stream) left: counters and flags start at zero
    FDAS_CUDA_TRY(p, cudaMemsetAsync(scratch, 0, sizeof(int) * (size_t)(FDAS_STATIC_CTR_INTS + tiles), st));
    fdas_search_args sa = {};
    sa.enabled = 1;
    sa.thr = threshold;
    sa.cand_span = 8;
    sa.tile_count = scratch;
    sa.tile_count_next = scratch + 1;
    sa.tile_flags = scratch + FDAS_STATIC_CTR_INTS;
    sa.tile_list = scratch + FDAS_STATIC_CTR_INTS + FDAS_STATIC_TILES;
    sa.scratch = nullptr;   // one template group: the recheck strip is in shared memory
    sa.peaks = peaks_dev;
    sa.capacity = capacity;
    sa.counts = count_dev;
    const TbMaps no_maps = {};   // neither launch stores through a tensor map

    TcParams tp;
    tc_fill_params(p, tp, spectrum_dev, nullptr, 1, R);
    tp.search = sa;
    const unsigned gx = fdas_tc_split_ctas(p, tp, tp.n_blocks);
    int rc = split == 3 ? launch_nch<3, TB_SCAN>(p, tp, gx, scan_smem, &no_maps, st) : launch_nch<1, TB_SCAN>(p, tp, gx, scan_smem, &no_maps, st);
    if (rc) return rc;
    tc_fill_params(p, tp, spectrum_dev, nullptr, 1, FDAS_TC_STRIP);
    tp.search = sa;
    tp.clustered = 0;
    const unsigned gr = (unsigned)(tiles < p->num_sms ? tiles : p->num_sms);
    return split == 3 ? launch_nch<3, TB_RECHECK>(p, tp, gr, recheck_smem, &no_maps, st) : launch_nch<1, TB_RECHECK>(p, tp, gr, recheck_smem, &no_maps, st);
}
