// fdas_mma.cu -- host side of the tensor-core form of the convolution (include/fdas.h: fdas_convolve with
// FDAS_ALGO_MMA, the default for FDAS_BF16 and FDAS_F32): |z| grouping, tap-matrix build, tensor maps, launch.
// The kernels and their design notes are in fdas_mma_kernels.cuh.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include "fdas_mma_kernels.cuh"

namespace {

// ---- tap matrix builder -----------------------------------------------------------------
// bmat[g][q][n][e], kappa = 8 q + e, j = M0 - kappa: bf16(RNE, once from fp64) of h_{+|z|}[j] for
// |z| index zi = g*nzg + 2 (n/4) + (n & 1), real part if (n & 2) == 0 else imaginary; zero padding.
// kref[g][zi] = (template whose fp64 taps are read, +1 if its z >= 0 else -1): h_{+|z|} = conj(h_{-|z|}).
// split != 0 (fp32 variant): the tap is rounded to fp32 first (that variant's storage type, A11) and
// image 0 holds h1 = bf16(h), image 1 (at bmat + total) h2 = bf16(h - h1).
__global__ void fdas_tapmatrix_kernel(__nv_bfloat16 *bmat, const double2 *__restrict__ taps, const int2 *__restrict__ kref,
                                      int groups, int nzg, int NT, int KS, int m_max, int split)
{
    const size_t total = (size_t)groups * 2 * KS * NT * 8;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int e = (int)(idx % 8);
        const int n = (int)((idx / 8) % NT);
        const int qq = (int)((idx / 8 / NT) % (2 * KS));
        const int g = (int)(idx / 8 / NT / (2 * KS));
        const int j = m_max - (8 * qq + e);
        const int zi = fdas_tc_entry_of_column(n);
        double v = 0.0;
        if (j >= -m_max && zi < nzg) {
            const int2 kr = kref[(size_t)g * nzg + zi];
            if (kr.x >= 0) {
                const double2 h = taps[(size_t)kr.x * (2 * m_max + 1) + (m_max + j)];
                v = fdas_tc_column_is_imag(n) ? (double)kr.y * h.y : h.x;
            }
        }
        if (!split) {
            bmat[idx] = __double2bfloat16(v);
        } else {
            const float vf = (float)v;
            const __nv_bfloat16 h1 = __float2bfloat16_rn(vf);
            bmat[idx] = h1;
            bmat[total + idx] = __float2bfloat16_rn(vf - __bfloat162float(h1));
        }
    }
}

}  // namespace

// Host: the |z| grouping.  Templates z_k = -zmax + k dz pair up as (k, K-1-k) when zmax is a
// multiple of dz; otherwise every template stands alone.
int fdas_mma_plan(fdas_plan *p)
{
    if (p->precision != FDAS_BF16 && p->precision != FDAS_F32) return FDAS_OK;
    const int K = p->K;
    const bool symmetric = fabs(-2.0 * p->zmax + (K - 1) * p->dz) <= 1e-9 * (1.0 + p->zmax);
    const int nz = symmetric ? (K + 1) / 2 : K;
    const int groups = (nz + 63) / 64;
    const int nzg = (nz + groups - 1) / groups;
    const int NT = (2 * nzg + 15) / 16 * 16;
    const int KS = (2 * p->m_max + 1 + 15) / 16;
    // row offsets k*M are 32-bit plane-element offsets inside the kernel
    p->tc_supported = (KS <= FDAS_TC_MAX_KS && NT <= 128 && (long long)K * p->M < 0xFFFFFFFFLL);
    // fp32 variant (two tap images, four Z parts): must fit shared memory at the smallest work item
    if (p->precision == FDAS_F32 && TbSmem(128, KS, NT, TC_TILE * 4, 3).total > 227u * 1024u) p->tc_supported = 0;
    p->tc_groups = groups;
    p->tc_nzg = nzg;
    p->tc_NT = NT;
    p->tc_KS = KS;
    if (!p->tc_supported) return FDAS_OK;
    const size_t n_tab = (size_t)groups * nzg;
    int2 *tab = (int2 *)malloc(n_tab * sizeof(int2));   // plane rows (+|z|, -|z|)
    int2 *ref = (int2 *)malloc(n_tab * sizeof(int2));   // (template to read taps from, its sign)
    if (!tab || !ref) {
        free(tab);
        free(ref);
        return FDAS_ERR_ALLOC;
    }
    for (size_t i = 0; i < n_tab; ++i) {
        tab[i] = make_int2(-1, -1);
        ref[i] = make_int2(-1, 1);
        if ((int)i >= nz) continue;
        if (symmetric) {
            // |z| descending: i = 0 is +-zmax; the last entry is z = 0 (its own mirror)
            const int kp = K - 1 - (int)i, kn = (int)i;
            tab[i] = make_int2(kp, kn);   // z = 0: both entries name the same row (equal values, V = 0)
            ref[i] = make_int2(kp, 1);
        } else {
            // no mirror pairs: every template is listed as the "-|z|" row of an entry whose columns
            // hold conj(h_z) (the -|z| row conjugates them again), so that the rows of consecutive
            // entries are consecutive plane rows
            tab[i] = make_int2(-1, (int)i);
            ref[i] = make_int2((int)i, -1);
        }
    }
    // columns each K step needs (symmetric grids: entries are in descending |z| = descending tap count, so a K
    // step whose taps j = m_max - 16 ks - 15 .. m_max - 16 ks lie beyond an entry's half-width multiplies zeros)
    for (int g = 0; g < 8; ++g) {
        p->tc_nks_lo[g] = p->tc_nks_hi[g] = 0;   // nibble 0 = full width
        p->tc_ks_first[g] = 0;
    }
    if (symmetric) {
        for (int g = 0; g < groups && g < 8; ++g) {
            for (int ks = 0; ks < KS; ++ks) {
                const int jhi = p->m_max - 16 * ks, jlo = jhi - 15;
                const int minabs = (jlo <= 0 && jhi >= 0) ? 0 : (abs(jlo) < abs(jhi) ? abs(jlo) : abs(jhi));
                int n_need = 0;
                for (int e = 0; e < nzg; ++e) {
                    const size_t i = (size_t)g * nzg + e;
                    if ((int)i >= nz) break;
                    const double z = -p->zmax + tab[i].y * p->dz;   // the -|z| member of the pair
                    const int m_e = (int)ceil(fabs(z) / 2.0 + fabs(p->jerk) / 12.0) + 16;
                    if (m_e >= minabs) n_need = e + 1;
                }
                int cols = 4 * ((n_need + 1) / 2);
                cols = (cols + 15) / 16 * 16;
                if (cols < 16) cols = 16;
                if (cols > NT) cols = NT;
                // nibble 15 (NT / 16 <= 8 leaves it free): no template of the group reaches this step
                const unsigned long long nib = n_need == 0 ? 15ull : (unsigned long long)(cols / 16);
                if (ks < 16) p->tc_nks_lo[g] |= nib << (4 * ks);
                else p->tc_nks_hi[g] |= nib << (4 * (ks - 16));
                if (minabs == 0) p->tc_ks_first[g] = ks;              // holds tap j = 0: every entry needs it
            }
        }
    }
    // the K steps in issue order: the full-width step first, then on through the taps, wrapping round; a step no
    // template of the group reaches (a group of narrow templates: its outer taps are all zero) is left out.  Table 8
    // serves the groups beyond the eighth: natural order, every step at full width.  tc_cost[g]: estimated tensor-pipe
    // cycles per 128-bin tile (an M = 128, K = 16 MMA costs max(51, (4 KB + 32 N B) / 113 B per cycle), measured).
    for (int g = 0; g < FDAS_TC_STEP_TABLES; ++g) {
        const bool own = g < 8 && g < groups && symmetric;
        int n = 0;
        double cost = 0.0;
        for (int i = 0; i < KS; ++i) {
            const int ks = ((own ? p->tc_ks_first[g] : 0) + i) % KS;
            unsigned nib = 0;
            if (own) {
                nib = (unsigned)((ks < 16 ? p->tc_nks_lo[g] >> (4 * ks) : p->tc_nks_hi[g] >> (4 * (ks - 16))) & 15ull);
                if (nib == 15u) continue;   // marked below: nobody reaches this step
            }
            const uint32_t cols = nib ? 16u * nib : (uint32_t)NT;
            p->tc_steps[g][n++] = tc_step_entry(cols, (uint32_t)ks, (uint32_t)NT);
            const double c = (4096.0 + 32.0 * cols) / 113.0;
            cost += 2.0 * (c > 51.0 ? c : 51.0);
        }
        for (int i = n; i < FDAS_TC_MAX_KS; ++i) p->tc_steps[g][i] = 0;
        p->tc_nsteps[g] = n;
        if (g < 8) {
            p->tc_cost[g] = cost;
            int rows = 0;
            for (int e = 0; e < nzg && g < groups; ++e) {
                const int2 t = tab[(size_t)g * nzg + e];
                rows += (t.y >= 0) + (t.x >= 0 && t.x != t.y);
            }
            p->tc_rows[g] = rows;
        }
    }
    // leading 16-column chunks (8 |z| each) in which every entry has both plane rows, in every group
    p->tc_full_chunks = NT / 16;
    for (int g = 0; g < groups; ++g) {
        int lead = 0;
        while (lead < nzg && tab[(size_t)g * nzg + lead].x >= 0 && tab[(size_t)g * nzg + lead].y >= 0) ++lead;
        if (lead / 8 < p->tc_full_chunks) p->tc_full_chunks = lead / 8;
    }
    // bulk kernel (fdas_mma_bulk_kernel): per (group, column group of 2 NCH entries) the runs of
    // consecutive plane rows its staging rows map to: -|z| rows of entries el = 0.. ascending,
    // +|z| rows ascending with el descending; a mirror entry (z = 0) keeps its -|z| listing only.
    const int EPC = NT / 8;   // entries per column group = 2 NCH
    int4 *rng = (int4 *)malloc((size_t)groups * 4 * sizeof(int4));
    if (!rng) {
        free(tab);
        free(ref);
        return FDAS_ERR_ALLOC;
    }
    p->tc_bulk_ok = 1;
    p->tc_n_boxes = 0;
    for (int g = 0; g < groups; ++g)
        for (int cg = 0; cg < 4; ++cg) {
            int4 r = make_int4(0, 0, 0, 0);
            int x0 = -1;
            for (int el = 0; el < EPC; ++el) {
                const int e = cg * EPC + el;
                const int2 t = e < nzg ? tab[(size_t)g * nzg + e] : make_int2(-1, -1);
                if (t.y >= 0) {
                    if (r.y == 0) r.x = t.y;
                    if (el != r.y || t.y != r.x + r.y) p->tc_bulk_ok = 0;
                    r.y += 1;
                }
                if (t.x >= 0 && t.x != t.y) {
                    if (r.w == 0) x0 = t.x;
                    if (el != r.w || t.x != x0 - r.w) p->tc_bulk_ok = 0;
                    r.w += 1;
                }
            }
            r.z = r.w > 0 ? x0 - (r.w - 1) : 0;
            // the run length picks the tensor map whose box has exactly that many rows (index in bits 16+)
            for (int *cnt : {&r.y, &r.w}) {
                if (*cnt == 0) continue;
                int b = 0;
                while (b < p->tc_n_boxes && p->tc_box_heights[b] != *cnt) ++b;
                if (b == p->tc_n_boxes) {
                    if (b == FDAS_TC_MAX_BOXES) {
                        p->tc_bulk_ok = 0;
                        continue;
                    }
                    p->tc_box_heights[p->tc_n_boxes++] = *cnt;
                }
                *cnt |= b << 16;
            }
            rng[g * 4 + cg] = r;
        }
    // one image [groups][2 KS][NT][8] bf16; the fp32 variant keeps two (h1, h2)
    p->tc_bmat_bytes = (size_t)groups * 2 * KS * NT * 16 * (p->precision == FDAS_F32 ? 2 : 1);
    cudaError_t e;
    if ((e = cudaMalloc(&p->tc_bmat, p->tc_bmat_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tc_ktab, n_tab * sizeof(int2))) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tc_kref, n_tab * sizeof(int2))) != cudaSuccess ||
        (e = cudaMemcpy(p->tc_ktab, tab, n_tab * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(p->tc_kref, ref, n_tab * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tc_ranges, (size_t)groups * 4 * sizeof(int4))) != cudaSuccess ||
        (e = cudaMemcpy(p->tc_ranges, rng, (size_t)groups * 4 * sizeof(int4), cudaMemcpyHostToDevice)) != cudaSuccess) {
        free(tab);
        free(ref);
        free(rng);
        p->last_err = e;
        return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
    }
    free(tab);
    free(ref);
    free(rng);
    return FDAS_OK;
}

int fdas_launch_build_tapmatrix(fdas_plan *p, cudaStream_t st)
{
    if ((p->precision != FDAS_BF16 && p->precision != FDAS_F32) || !p->tc_supported) return FDAS_OK;
    const int split = p->precision == FDAS_F32;
    const size_t total = p->tc_bmat_bytes / 2 / (split ? 2 : 1);
    const int blocks = (int)((total + 255) / 256 < 1024 ? (total + 255) / 256 : 1024);
    fdas_tapmatrix_kernel<<<blocks, 256, 0, st>>>((__nv_bfloat16 *)p->tc_bmat, p->taps, p->tc_kref,
                                                  p->tc_groups, p->tc_nzg, p->tc_NT, p->tc_KS, p->m_max, split);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

// The planes as a rank-2 fp32 tensor [batch*K rows][M bins] with one box shape per distinct run
// length (tc_box_heights[] rows x 128 bins), for the bulk kernel's stores.  Encoded on the host (cuTensorMapEncodeTiled, fetched through
// the runtime so that libfdas does not link libcuda) and cached for the last plane buffer.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int fdas_tc_encode_maps(fdas_plan *p, void *base, long long cols, long long rows, size_t elem_bytes, void *maps_out)
{
    static EncodeTiledFn encode = nullptr;   // a driver entry point: the same for every device and thread
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        FDAS_CUDA_TRY(p, cudaGetDriverEntryPointByVersion("cuTensorMapEncodeTiled", &fn, 12000, cudaEnableDefault, &qres));
        if (!fn || qres != cudaDriverEntryPointSuccess) return FDAS_ERR_UNSUPPORTED;
        encode = (EncodeTiledFn)fn;
    }
    TbMaps *maps = static_cast<TbMaps *>(maps_out);
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)cols * elem_bytes};
    const cuuint32_t estr[2] = {1, 1};
    for (int b = 0; b < p->tc_n_boxes; ++b) {
        const cuuint32_t box[2] = {(cuuint32_t)TC_TILE, (cuuint32_t)p->tc_box_heights[b]};
        const CUresult r = encode(&maps->m[b], elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                                  base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                  CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return FDAS_ERR_UNSUPPORTED;
    }
    return FDAS_OK;
}

static int plane_maps(fdas_plan *p, void *planes, int batch, const TbMaps **out)
{
    if (!p->tc_maps) {
        p->tc_maps = aligned_alloc(64, sizeof(TbMaps));
        if (!p->tc_maps) return FDAS_ERR_ALLOC;
        p->tc_maps_plane = nullptr;
    }
    const size_t esz = p->plane_bf16 ? 2 : 4;
    if (p->tc_maps_plane != planes || p->tc_maps_batch != batch || p->tc_maps_elem != (int)esz) {
        p->tc_maps_plane = nullptr;
        const int rc = fdas_tc_encode_maps(p, planes, p->M, (long long)batch * p->K, esz, p->tc_maps);
        if (rc != FDAS_OK) return rc;
        p->tc_maps_plane = planes;
        p->tc_maps_batch = batch;
        p->tc_maps_elem = (int)esz;
    }
    *out = static_cast<TbMaps *>(p->tc_maps);
    return FDAS_OK;
}

template <int NCH>
static int launch_mma_split(fdas_plan *p, const TcParams &tp, unsigned gx, size_t smem_bytes, const TbMaps *maps, cudaStream_t st)
{
    auto kern = fdas_mma_bulk_kernel<NCH, float, 3>;
    { const int rc = fdas_optin_smem(p, FDAS_OPTIN_MMA_SPLIT, kern, smem_bytes); if (rc) return rc; }
    kern<<<dim3(gx), tb_threads(3), smem_bytes, st>>>(tp, *maps);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

template <int NCH, typename OT>
static int launch_mma(fdas_plan *p, const TcParams &tp, unsigned gx, size_t smem_bytes, const TbMaps *maps, cudaStream_t st)
{
    if (maps) {
        auto kern = fdas_mma_bulk_kernel<NCH, OT, 1>;
        { const int rc = fdas_optin_smem(p, sizeof(OT) == 2 ? FDAS_OPTIN_MMA_BULK16 : FDAS_OPTIN_MMA_BULK, kern, smem_bytes); if (rc) return rc; }
        kern<<<dim3(gx), tb_threads(1), smem_bytes, st>>>(tp, *maps);
    } else {
        auto kern = fdas_mma_convolve_kernel<NCH, OT>;
        { const int rc = fdas_optin_smem(p, sizeof(OT) == 2 ? FDAS_OPTIN_MMA_SCALAR16 : FDAS_OPTIN_MMA_SCALAR, kern, smem_bytes); if (rc) return rc; }
        kern<<<dim3(gx), TC_THREADS, smem_bytes, st>>>(tp);
    }
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

// What fdas_launch_convolve_mma launches for (plane buffer, batch): decided once, used by the launch and by
// fdas_describe_convolve.
struct TcDecision {
    bool bulk;          // box stores through tensor maps (fdas_mma_bulk_kernel) or per-thread stores (fdas_mma_convolve_kernel)
    int split;          // 1: bf16 operands; 3: fp32 operands split into bf16 terms
    int R;              // bins per work item
    uint32_t smem;      // dynamic shared memory
    unsigned gx;        // CTAs per template group
    const TbMaps *maps;
};

static int tc_decide(fdas_plan *p, void *planes, int batch, bool want_maps, TcDecision &d)
{
    if ((p->precision != FDAS_BF16 && p->precision != FDAS_F32) || !p->tc_supported) return FDAS_ERR_UNSUPPORTED;
    d.split = p->precision == FDAS_F32 ? 3 : 1;
    // tensor-map stores need 16-byte aligned plane rows: M % 4 == 0 (% 8 for a bf16 plane) and a 16-byte aligned plane
    const uint32_t esz = p->plane_bf16 ? 2u : 4u;
    d.bulk = ((p->M * esz) % 16 == 0) && ((reinterpret_cast<uintptr_t>(planes) & 15u) == 0) && !p->tc_force_scalar_stores &&
             p->tc_bulk_ok && (long long)batch * p->K < 0x7FFFFFFFLL;
    d.maps = nullptr;
    if (d.bulk && want_maps && plane_maps(p, planes, batch, &d.maps) != FDAS_OK) {   // no encoder in this driver: scalar stores
        d.bulk = false;
        d.maps = nullptr;
    }
    if (d.split == 3 && !d.bulk) return FDAS_ERR_UNSUPPORTED;   // the split-operand form exists with box stores only
    const uint32_t smem_cap = 227u * 1024u;
    auto smem_total = [&](int R) -> uint32_t {
        return d.bulk ? TbSmem(R, p->tc_KS, p->tc_NT, TC_TILE * esz, d.split).total : TcSmem(R, p->tc_KS, p->tc_NT).total;
    };
    // outputs per work item: the largest of 1024..128 that fits shared memory and leaves at
    // least two items per CTA
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    int R = 1024;
    for (;; R >>= 1) {
        const long long items = (long long)batch * ((p->M + R - 1) / R);
        if (R == 128 || (smem_total(R) <= smem_cap && items >= 2LL * sms_per_group)) break;
    }
    R = fdas_tc_balance_items(R, p->M, batch, sms_per_group);
    d.R = R;
    d.smem = smem_total(R);
    if (d.smem > smem_cap) return FDAS_ERR_UNSUPPORTED;
    const long long items = (long long)batch * ((p->M + R - 1) / R);
    if (items >= 0x7FFFFFFFLL) return FDAS_ERR_UNSUPPORTED;   // the kernels count work items in 32 bits
    d.gx = (unsigned)(items < sms_per_group ? items : sms_per_group);
    return FDAS_OK;
}

// Does a launch skip, per K step, the columns no template of that step reaches (exact zeros; the sums do not change)?
// Always where the tensor pipe bounds the launch: the split-operand form, the plane-free search, the bf16-stored
// plane.  A float plane with bf16 operands is bound by its stores when the MMA stream is short against them --
// config 3 (97 templates, 9 K steps) measured 0.297 ms at full width against 0.309 ms trimmed -- and by the SM side
// when it is not -- config 5 (201 templates in two groups, 15 K steps): 0.781 ms at full width, 0.734 ms trimmed.
// The rule between the two: MMA cycles per 128-bin tile (groups x 2 KS x ~66) against the cycles the tile's K rows of
// 512 bytes take at the store rate of one SM's share (~25 per row); trimmed above 0.6.
int fdas_tc_trims(const fdas_plan *p, bool plane_free)
{
    if (p->precision == FDAS_F32 || plane_free || p->plane_bf16) return 1;
    const double mma = (double)p->tc_groups * 2.0 * p->tc_KS * 66.0, store = 25.0 * p->K;
    return mma > 0.6 * store;
}

// dense MMA flops one launch over `batch` series issues (padding included): per 128-bin tile and template group,
// 2 parts x sum over the K steps of 2 * 128 * N_ks * 16, three products per tap in the split form; plane_free: the
// scan launch of the plane-free search
double fdas_tc_issued_flops(const fdas_plan *p, int batch, int plane_free)
{
    const int split = p->precision == FDAS_F32 ? 3 : 1;
    const bool trimmed = fdas_tc_trims(p, plane_free != 0);
    double per_tile = 0.0;
    for (int g = 0; g < p->tc_groups; ++g) {
        const int tb = g < FDAS_TC_STEP_TABLES - 1 ? g : FDAS_TC_STEP_TABLES - 1;
        for (int i = 0; i < p->tc_nsteps[tb]; ++i) {
            const int n = trimmed ? (int)(((uint32_t)p->tc_steps[tb][i] >> 17) & 63u) * 8 : p->tc_NT;   // N field of the descriptor
            per_tile += 2.0 * 2.0 * TC_TILE * n * 16.0 * (split == 3 ? 3.0 : 1.0);
        }
    }
    return per_tile * (double)batch * (double)((p->M + TC_TILE - 1) / TC_TILE);
}

int fdas_tc_describe(fdas_plan *p, const void *plane_dev, int batch, fdas_kernel_info_t *out)
{
    TcDecision d;
    const int rc = tc_decide(p, const_cast<void *>(plane_dev), batch, false, d);
    if (rc) return rc;
    out->algorithm = d.bulk ? FDAS_ALGO_MMA : FDAS_ALGO_MMA_SCALAR;
    out->split = d.split;
    out->groups = p->tc_groups;
    out->nch = p->tc_NT / 16;
    out->k_steps = p->tc_KS;
    out->work_item_bins = d.R;
    {
        TcParams tp;
        tc_fill_params(p, tp, nullptr, const_cast<void *>(plane_dev), batch, d.R);
        out->grid_x = (int32_t)fdas_tc_split_ctas(p, tp, (long long)batch * tp.n_blocks);   // one-dimensional: every group's CTAs
        out->grid_y = 1;
    }
    out->block_threads = d.bulk ? tb_threads(d.split) : TC_THREADS;
    out->dynamic_smem_bytes = d.smem;
    out->tensor_flops = fdas_tc_issued_flops(p, batch, 0);
    if (d.bulk)
        snprintf(out->kernel, sizeof(out->kernel), "fdas_mma_bulk_kernel<%d, %s, %d>", p->tc_NT / 16, p->plane_bf16 ? "__nv_bfloat16" : "float", d.split);
    else
        snprintf(out->kernel, sizeof(out->kernel), "fdas_mma_convolve_kernel<%d, %s>", p->tc_NT / 16, p->plane_bf16 ? "__nv_bfloat16" : "float");
    return FDAS_OK;
}

int fdas_launch_convolve_mma(fdas_plan *p, const void *spectra, void *planes, int batch, cudaStream_t st,
                             fdas_search_args *search)
{
    TcDecision d;
    { const int rc = tc_decide(p, planes, batch, true, d); if (rc) return rc; }
    const bool bulk = d.bulk;
    const int split = d.split, R = d.R;
    const uint32_t total = d.smem;
    const TbMaps *maps = d.maps;
    TcParams tp;
    tc_fill_params(p, tp, spectra, planes, batch, R);
    const unsigned gx = fdas_tc_split_ctas(p, tp, (long long)batch * tp.n_blocks);   // all CTAs, every group
    if (search) {
        search->cand_span = bulk ? p->tc_NT / 8 : 8;   // |z| entries per column group (2 NCH) / per 16-column chunk
        tp.search = *search;
    } else {
        tp.search = fdas_search_args{};
        tp.search.cand_span = 8;
    }
    switch (p->tc_NT / 16) {
    case 1: if (split == 3) return launch_mma_split<1>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<1, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<1, float>(p, tp, gx, total, maps, st);
    case 2: if (split == 3) return launch_mma_split<2>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<2, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<2, float>(p, tp, gx, total, maps, st);
    case 3: if (split == 3) return launch_mma_split<3>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<3, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<3, float>(p, tp, gx, total, maps, st);
    case 4: if (split == 3) return launch_mma_split<4>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<4, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<4, float>(p, tp, gx, total, maps, st);
    case 5: if (split == 3) return launch_mma_split<5>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<5, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<5, float>(p, tp, gx, total, maps, st);
    case 6: if (split == 3) return launch_mma_split<6>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<6, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<6, float>(p, tp, gx, total, maps, st);
    case 7: if (split == 3) return launch_mma_split<7>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<7, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<7, float>(p, tp, gx, total, maps, st);
    case 8: if (split == 3) return launch_mma_split<8>(p, tp, gx, total, maps, st);
            return p->plane_bf16 ? launch_mma<8, __nv_bfloat16>(p, tp, gx, total, maps, st) : launch_mma<8, float>(p, tp, gx, total, maps, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}
