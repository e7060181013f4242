// fdas_mma_kernels.cuh -- device code of the tensor-core (tcgen05 / TMEM) form of the convolution, shared by
// fdas_mma.cu (fdas_convolve, fdas_search with a plane) and fdas_mma_search.cu (plane-free fdas_search).
//
//
// the f-fdot plane is the spectrum convolved with every template,
//      Y_z[r] = sum_{j=-m_z..m_z} X[r-j] h_z[j],   P[k][r] = |Y_{z_k}[r]|^2 .
// PAPER.md:65-67 computes that linear convolution by overlap-save FFTs because on the
// hardware the paper names a 2 m + 1 <= 129 tap complex filter bank is cheaper through FFTs.
// On B200 the same sum is a dense contraction the 5th-generation tensor cores finish faster
// than the FFT butterflies run on the fp32 ALUs, with bf16 operands
// and fp32 accumulation -- "bf16 storage / fp32 accumulate" literally:
//
//      D[r][n] = sum_kappa T[r][kappa] * B[n][kappa]
//      T[r][kappa] = X_part[r - M0 + kappa]      (Toeplitz matrix of the spectrum, part = re | im)
//      B[n][kappa] = hre_|z|[M0 - kappa] or him_|z|[M0 - kappa]; the columns of two consecutive
//                    |z| entries e, e+1 are ordered (hre_e, hre_e+1, him_e, him_e+1) so that
//                    the accumulators of an entry pair sit in adjacent registers (packed
//                    fp32x2 arithmetic in the epilogue)
//
// The Toeplitz matrix is never materialised per tile: shared memory holds Z[i] = the eight
// consecutive bf16 samples X_part[g0 + i .. g0 + i + 7] as one 16-byte row, and a K-major,
// non-swizzled UMMA descriptor with leading- and stride-byte-offset both 128 B makes core
// matrix (row group g, K chunk c) start at Z row 8 (g + c): consecutive tiles, K steps and
// row groups all alias the same rows of Z.
//
// Symmetry h_{-z} = conj(h_z) (DESIGN.md pin P3) halves the contraction: with real filters
// hre, him of +|z| and U = X * hre, V = X * him (complex X, so Ure, Uim, Vre, Vim),
//      Y_{+|z|} = (Ure - Vim) + i (Uim + Vre),     Y_{-|z|} = (Ure + Vim) + i (Uim - Vre).
// Two MMAs per K step (A = Toeplitz of re(X), of im(X); same B) leave, for output r, Ure/Vre
// and Uim/Vim in the SAME TMEM lane, so the epilogue thread of lane r forms both powers
// without any exchange and a warp stores 32 consecutive bins of one plane row (128 bytes).
//
// One persistent CTA per SM, warp-specialised.  Two kernels share the loader and the MMA issuer:
//
// fdas_mma_bulk_kernel (M % 4 == 0, the normal case)
//   warps 0-15  epilogue, two sets taking alternate tiles: tcgen05.ld -> packed |.|^2, the powers
//               of the whole tile held in registers and the TMEM stage handed back at once, so
//               the MMAs never wait for the store path; then registers -> shared-memory staging
//               rows of 128 bins -> one tensor-map box store (cp.async.bulk.tensor.2d) per run of
//               consecutive plane rows.  Measured on B200: plane rows
//               written as 128-byte segments cap at ~4.5 TB/s, 256..1024-byte segments reach
//               5.8-6.0 TB/s, a linear fill 7.1 TB/s.
//   warp  16    one thread issues tcgen05.mma and tcgen05.commit
//   warps 17-19 loader: spectrum block -> bf16 (RNE, reading A12) -> Z rows
//
// Template parameters of fdas_mma_bulk_kernel: NCH (16-column chunks of the tap matrix), OT (plane
// element: float, or __nv_bfloat16 for the bf16-stored plane of PAPER.md:91), SPLIT (1: bf16 operands;
// 3: the fp32 variant -- x = x1 + x2 and h = h1 + h2 in bf16 terms, products x1 h1 + x1 h2 + x2 h1
// accumulated into the same TMEM columns, four Z parts, two tap images, ONE epilogue warp set).
// The taps may carry a jerk (fdas_plan_create_jerk): h_{-z,w} = conj h_{z,w} keeps the +-|z| pairing.
//
// fdas_mma_convolve_kernel (any M: bulk copies need 16-byte aligned rows)
//   warps 0-7   epilogue: tcgen05.ld -> |.|^2 -> st.global.cs (TMEM double-buffered)
//   warp  8     MMA issuer;  warps 9-11 loader
#pragma once
#include <cuda.h>        // CUtensorMap (types only; the encoder is fetched through cudaGetDriverEntryPoint)
#include <cuda_bf16.h>
#include "fdas_internal.h"

namespace {


constexpr int TC_TILE = 128;            // outputs per MMA tile = UMMA M = TMEM lanes
constexpr int TC_EPI_WARPS = 8;
constexpr int TC_MMA_WARP = 8;
constexpr int TC_LOAD_WARP0 = 9;
constexpr int TC_LOAD_WARPS = 3;       // 16 + 1 + 3 = 20 warps: registers are granted per 4 warps, 20 warps leave 96 per thread
constexpr int TC_LOAD_THREADS = 32 * TC_LOAD_WARPS;
constexpr int TC_THREADS = 32 * (TC_EPI_WARPS + 1 + TC_LOAD_WARPS);   // 384
constexpr int TC_TMEM_COLS = 512;       // whole TMEM: 2 stages x (re | im) x NT <= 128 columns
constexpr int TC_STAGE_COLS = 256;
#ifdef FDAS_SPIN_TRAP   // debug builds only (-DFDAS_SPIN_TRAP): a stuck pipeline traps instead of hanging the GPU
constexpr long long TC_SPIN_LIMIT = 1LL << 26;
#endif

// tcgen05 instruction descriptor (cute::UMMA::InstrDescriptor): fp32 accumulate, bf16 A and B, both K-major, M = 128,
// N = n_cols (a multiple of 16)
__host__ __device__ constexpr uint32_t tc_idesc(uint32_t n_cols)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(TC_TILE >> 4) << 24) | ((n_cols >> 3) << 17);
}
// one K step of the issue order: bits 0-31 the instruction descriptor (N = the columns whose templates reach the
// step), bits 32-47 the offset of the step's Z rows, bits 48-63 the offset of its tap chunk pair, both in units of
// 16 bytes (what a shared-memory descriptor's address field counts)
__host__ __device__ constexpr unsigned long long tc_step_entry(uint32_t n_cols, uint32_t ks, uint32_t NT)
{
    return (unsigned long long)tc_idesc(n_cols) | ((unsigned long long)(ks * 16u) << 32) |
           ((unsigned long long)(ks * 2u * NT) << 48);
}

struct TcParams {
    const float2 *spectra;   // [batch][M] complex64
    void *planes;            // [batch][K][M] float, or bf16 bit patterns when the plan stores a bf16 plane
    const uint4 *bmat;       // [groups][2 KS][NT] rows of 8 bf16 (the shared-memory image)
    const int2 *ktab;        // [groups][nzg]: plane rows of (+|z|, -|z|), -1 where absent
    const int4 *ranges;      // bulk kernel: [groups][4 column groups] (row0_n, cnt_n, row0_p, cnt_p), see fdas_mma_plan
    long long M;
    int K, batch;
    int R;                   // outputs per work item (multiple of 128)
    int n_blocks;            // work items per series in this launch: ceil(M / R), or the blocks of a bin range
    int blk_first;           // first block of that range (0: the whole series)
    int M0;                  // m_max: T[r][kappa] = X[r - M0 + kappa]
    int KS;                  // K steps of 16 taps
    int NT;                  // UMMA N: columns per part (multiple of 16, <= 128) = 16 NCH
    int nzg;                 // |z| values per group
    int full_chunks;         // 16-column chunks whose 8 |z| entries all have both plane rows
    // K steps in issue order, per template group (the first 8 groups; the others use row 8: every step at full width):
    // tc_step_entry(instruction descriptor with the columns the step needs, offset of its A rows, offset of its tap
    // chunk).  Read through the constant bank with a uniform index: the MMA warp never leaves the uniform datapath.
    unsigned long long steps[FDAS_TC_STEP_TABLES][FDAS_TC_MAX_KS];
    int nsteps[FDAS_TC_STEP_TABLES];   // entries of steps[g]: the K steps at least one template of the group reaches
    // CTA -> (template group, index inside the group).  TB_PLANE / TB_SCAN launches use a one-dimensional grid: with up
    // to 8 groups, group g owns CTAs cta0[g] .. cta0[g + 1] - 1, as many as its share of the MMA work (a group of narrow
    // templates needs fewer K steps per tile; fdas_tc_split_ctas); with more groups cta_even CTAs each.  TB_RECHECK
    // launches keep the grid (x, groups): the groups of one item form a cluster.
    int groups, cta_even;
    int cta0[FDAS_TC_STEP_TABLES];
    int trim;                // K steps skip the columns no template of theirs reaches (fdas_tc_trims)
    int tiles_per_series;    // ceil(M / 128): plane-free search numbers the tiles series * tiles_per_series + tile
    int clustered;           // recheck launch with more than one template group: the groups of one item form a cluster
    fdas_search_args search; // fused threshold pass (fdas_search); enabled = 0 for plain fdas_convolve
};

// host: everything of TcParams that follows from the plan and the work-item size R (search left disabled)
static inline void tc_fill_params(const fdas_plan *p, TcParams &tp, const void *spectra, void *planes, int batch, int R)
{
    tp.spectra = static_cast<const float2 *>(spectra);
    tp.planes = planes;
    tp.bmat = static_cast<const uint4 *>(p->tc_bmat);
    tp.ktab = p->tc_ktab;
    tp.ranges = p->tc_ranges;
    tp.M = p->M;
    tp.K = p->K;
    tp.batch = batch;
    tp.R = R;
    tp.n_blocks = (int)((p->M + R - 1) / R);
    tp.blk_first = 0;
    tp.M0 = p->m_max;
    tp.KS = p->tc_KS;
    tp.NT = p->tc_NT;
    tp.nzg = p->tc_nzg;
    tp.full_chunks = p->tc_full_chunks;
    for (int g = 0; g < FDAS_TC_STEP_TABLES; ++g) {
        for (int i = 0; i < FDAS_TC_MAX_KS; ++i) tp.steps[g][i] = p->tc_steps[g][i];
        tp.nsteps[g] = p->tc_nsteps[g];
        tp.cta0[g] = 0;
    }
    tp.groups = p->tc_groups;
    tp.cta_even = 1;
    tp.trim = fdas_tc_trims(p, planes == nullptr);
    tp.tiles_per_series = (int)((p->M + 127) / 128);
    tp.clustered = 0;
    tp.search = fdas_search_args{};
    tp.search.cand_span = 8;
}

// Work-item size against the tail: with a handful of items per CTA the CTAs holding one item more than the others set
// the launch time (config 2: 512 items of 1024 bins on 148 CTAs = 4 rounds where 3.46 would do).  Halving the item (at
// most twice, never below 128 bins) is taken when it shortens the longest CTA's share of bins by 8 % or more; long
// launches keep the largest item (fewer halo rows to load, the store pattern measured fastest).
static inline int fdas_tc_balance_items(int R, long long M, int batch, int ctas)
{
    auto share = [&](int r) {
        const long long items = (long long)batch * ((M + r - 1) / r);
        return ((items + ctas - 1) / ctas) * r;
    };
    int best = R;
    for (int r = R >> 1, n = 0; r >= 128 && n < 2; r >>= 1, ++n)
        if (share(r) * 100 <= share(best) * 92) best = r;
    return best;
}

// CTAs of a TB_PLANE / TB_SCAN launch over `items` work items per template group: total returned, tp.cta0 / cta_even
// filled.  Up to 8 groups share the SMs in proportion to their cost per tile (tensor work or plane stores, whichever
// bounds the group), at least one CTA and at most `items` each; more groups get the same number each.
static inline unsigned fdas_tc_split_ctas(const fdas_plan *p, TcParams &tp, long long items)
{
    const int G = p->tc_groups;
    const int even = p->num_sms / G > 0 ? p->num_sms / G : 1;
    tp.cta_even = (int)(items < even ? items : even);
    if (G > FDAS_TC_STEP_TABLES - 1) return (unsigned)tp.cta_even * (unsigned)G;
    // cost of a tile: its MMAs (three products per tap in the split form) or, if that takes longer, its plane rows at
    // one SM's share of the store rate (~25 cycles per 512-byte row segment: config 3 is store-bound at 97 rows in
    // 2400 cycles); a plane-free launch stores nothing
    const double per_row = tp.planes ? (p->plane_bf16 ? 12.5 : 25.0) : 0.0, products = p->precision == FDAS_F32 ? 3.0 : 1.0;
    double cost[FDAS_TC_STEP_TABLES - 1], total = 0.0;
    for (int g = 0; g < G; ++g) {
        const double mma = products * p->tc_cost[g], store = per_row * p->tc_rows[g];
        cost[g] = mma > store ? mma : store;
        total += cost[g];
    }
    int n[FDAS_TC_STEP_TABLES - 1], sum = 0;
    for (int g = 0; g < G; ++g) {
        n[g] = (int)(p->num_sms * cost[g] / total);
        if (n[g] < 1) n[g] = 1;
        sum += n[g];
    }
    for (int g = 0; sum < p->num_sms && G <= p->num_sms; g = (g + 1) % G, ++sum) n[g] += 1;   // rounding leftovers
    for (int g = 0; sum > p->num_sms && g < G; ++g)
        while (n[g] > 1 && sum > p->num_sms) { n[g] -= 1; sum -= 1; }
    tp.cta0[0] = 0;
    for (int g = 0; g < G; ++g) {
        if (n[g] > items) n[g] = (int)items;
        tp.cta0[g + 1] = tp.cta0[g] + n[g];
    }
    return (unsigned)tp.cta0[G];
}

// What a launch of fdas_mma_bulk_kernel does with the powers (template parameter MODE):
//   TB_PLANE    writes the plane (fdas_convolve; fdas_search with a plane also flags candidate cells)
//   TB_SCAN     plane-free search, first launch: no stores at all; flags the 128-bin tiles holding a power above the
//               threshold (search.tile_flags / tile_list)
//   TB_RECHECK  plane-free search, second launch: work items are the flagged tiles (with the neighbour tile where the
//               first / last bin is a candidate); the same MMAs and the same epilogue arithmetic recompute them --
//               bit-identical to what TB_PLANE stores -- into a private strip of scratch memory, then the epilogue
//               warps apply the peak rule of fdas_peaks to the cells of the flagged tile
constexpr int TB_PLANE = 0, TB_SCAN = 1, TB_RECHECK = 2;

// work item -> (series, first bin, tiles, index of the tile whose cells are tested [TB_RECHECK])
template <int MODE>
__device__ __forceinline__ void tb_item(const TcParams &p, uint32_t it, long long &ser, long long &blk0, int &n_tiles, int &centre)
{
    if constexpr (MODE == TB_RECHECK) {
        const int tg = __ldcg(p.search.tile_list + it);
        const int fl = __ldcg(p.search.tile_flags + tg);
        const int t = tg % p.tiles_per_series;
        ser = tg / p.tiles_per_series;
        const int hl = ((fl & 2) && t > 0) ? 1 : 0, hr = ((fl & 4) && t + 1 < p.tiles_per_series) ? 1 : 0;
        blk0 = (long long)(t - hl) * 128;
        n_tiles = 1 + hl + hr;
        centre = hl;
    } else {
        ser = it / (uint32_t)p.n_blocks;   // 32-bit division: items < 2^31 (checked by the launcher)
        blk0 = (long long)(p.blk_first + it % (uint32_t)p.n_blocks) * p.R;
        const long long left = p.M - blk0;
        n_tiles = (int)((left < p.R ? left : p.R) + 128 - 1) / 128;
        centre = 0;
    }
}
// work items of this launch
template <int MODE>
__device__ __forceinline__ uint32_t tb_items(const TcParams &p)
{
    if constexpr (MODE == TB_RECHECK) {
        const long long all = (long long)p.batch * p.tiles_per_series;
        const long long n = __ldcg(p.search.tile_count);
        return (uint32_t)(n < all ? n : all);
    } else {
        return (uint32_t)p.batch * (uint32_t)p.n_blocks;
    }
}
// This CTA's template group, its index among the CTAs of that group and their number (TcParams::cta0).  Only the
// group is kept in a register: x and nx are re-read from the constant bank where they are used (once per work item) --
// held in registers they cost the float-plane kernel a spill in its epilogue (96-register cap; 0.300 -> 0.309 ms).
struct TbCta {
    int grp;
    template <int MODE>
    __device__ __forceinline__ uint32_t x(const TcParams &p) const
    {
        if constexpr (MODE == TB_RECHECK) return blockIdx.x;
        else if (p.groups <= FDAS_TC_STEP_TABLES - 1) return blockIdx.x - (uint32_t)p.cta0[grp];
        else return blockIdx.x % (uint32_t)p.cta_even;
    }
    template <int MODE>
    __device__ __forceinline__ uint32_t nx(const TcParams &p) const
    {
        if constexpr (MODE == TB_RECHECK) return gridDim.x;
        else if (p.groups <= FDAS_TC_STEP_TABLES - 1) return (uint32_t)(p.cta0[grp + 1] - p.cta0[grp]);
        else return (uint32_t)p.cta_even;
    }
};
template <int MODE>
__device__ __forceinline__ TbCta tb_cta(const TcParams &p)
{
    TbCta c;
    if constexpr (MODE == TB_RECHECK) {
        c.grp = (int)blockIdx.y;
    } else if (p.groups <= FDAS_TC_STEP_TABLES - 1) {
        int g = 0;
        while (g + 1 < p.groups && (int)blockIdx.x >= p.cta0[g + 1]) ++g;
        c.grp = g;
    } else {
        c.grp = (int)(blockIdx.x / (uint32_t)p.cta_even);
    }
    return c;
}
// TB_RECHECK: the epilogue threads meet here twice per work item: once when the item's powers are in scratch, once
// when they have been tested.  One template group: a named barrier over the epilogue warps only, so the loader and
// the MMA warp run ahead into the next item.  Several groups (one CTA each, forming a cluster): a cluster barrier,
// which counts EVERY thread of the cluster -- the loader and MMA warps then call this too.
__device__ __forceinline__ void tb_item_sync(int clustered, int threads)
{
    __syncwarp();
    if (clustered) asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    else asm volatile("bar.sync 7, %0;" ::"r"(threads) : "memory");
}

// ---- PTX wrappers ---------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
template <int SLEEP_NS = 0>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t done;
#ifdef FDAS_SPIN_TRAP
    long long spins = 0;
#endif
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.b32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (!done) {
#ifdef FDAS_SPIN_TRAP
            if (++spins > TC_SPIN_LIMIT) __trap();
#endif
            if (SLEEP_NS > 0) __nanosleep(SLEEP_NS);
        }
    } while (!done);
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t holder_smem, uint32_t cols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(holder_smem), "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}

// TMEM -> registers: this warp's 32 lanes x 16 columns at taddr_a (v[0..15]) and at taddr_b
// (v[16..31]).  Asynchronous: v[] is defined only after tmem_ld_wait(v), which names the same
// registers as in/out operands so that no use can be scheduled before tcgen05.wait::ld.
__device__ __forceinline__ void tmem_ld32(uint32_t taddr_a, uint32_t taddr_b, uint32_t *v)
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%32];\n\t"
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%33];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr_a), "r"(taddr_b)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait(uint32_t *v)
{
    asm volatile(
        "tcgen05.wait::ld.sync.aligned;"
        : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3]), "+r"(v[4]), "+r"(v[5]), "+r"(v[6]), "+r"(v[7]),
          "+r"(v[8]), "+r"(v[9]), "+r"(v[10]), "+r"(v[11]), "+r"(v[12]), "+r"(v[13]), "+r"(v[14]), "+r"(v[15]),
          "+r"(v[16]), "+r"(v[17]), "+r"(v[18]), "+r"(v[19]), "+r"(v[20]), "+r"(v[21]), "+r"(v[22]), "+r"(v[23]),
          "+r"(v[24]), "+r"(v[25]), "+r"(v[26]), "+r"(v[27]), "+r"(v[28]), "+r"(v[29]), "+r"(v[30]), "+r"(v[31])
        :
        : "memory");
}

// K-major, non-swizzled shared-memory matrix descriptor (cute::UMMA::SmemDescriptor layout):
// bits [0,14) address >> 4, [16,30) leading byte offset >> 4 (between the two 8-element K
// chunks of one MMA), [32,46) stride byte offset >> 4 (between 8-row groups), bit 46 version.
// Held as two words: every operand of these kernels has stride byte offset 128 (consecutive 8-row groups are adjacent),
// so the high word is one constant and the low word carries the address and the leading byte offset
constexpr uint32_t TC_DESC_HI = (128u >> 4) | (1u << 14);
__device__ __forceinline__ uint32_t smem_desc_lo(uint32_t addr, uint32_t lbo_bytes)
{
    return ((addr >> 4) & 0x3FFFu) | (((lbo_bytes >> 4) & 0x3FFFu) << 16);
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);   // .x (low half) = lo
    return *reinterpret_cast<uint32_t *>(&v);
}

// shared-memory carve-up (bytes), the same arithmetic on host and device
struct TcSmem {
    uint32_t b_bytes, zr, z_part_bytes, z_buf_bytes, xn, xs_part_bytes;
    uint32_t off_z, off_xs, off_ktab, off_bars, off_holder, total;
    __host__ __device__ TcSmem(int R, int KS, int NT)
    {
        const uint32_t TP = 16u * KS;
        b_bytes = 2u * KS * NT * 16u;
        zr = R + TP - 8;
        z_part_bytes = zr * 16u;
        z_buf_bytes = 2u * z_part_bytes;
        xn = R + TP;
        xs_part_bytes = xn * 2u;
        off_z = b_bytes;
        off_xs = off_z + 2u * z_buf_bytes;
        off_ktab = (off_xs + 2u * xs_part_bytes + 15u) & ~15u;
        off_bars = (off_ktab + 8u * (NT / 2) + 15u) & ~15u;
        off_holder = off_bars + 8u * 8u;
        total = off_holder + 16u;
    }
};

// streaming store of v at base + off (plane elements): one IMAD.WIDE for the address.  OT = float, or
// __nv_bfloat16 for the bf16-stored plane of PAPER.md:91 (the power rounded once, RNE).
template <typename OT>
__device__ __forceinline__ void st_cs_at(const OT *base, uint32_t off, float v)
{
    unsigned long long addr;
    if constexpr (sizeof(OT) == 4) {
        asm("mad.wide.u32 %0, %1, 4, %2;" : "=l"(addr) : "r"(off), "l"(base));
        asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
    } else {
        asm("mad.wide.u32 %0, %1, 2, %2;" : "=l"(addr) : "r"(off), "l"(base));
        asm volatile("st.global.cs.u16 [%0], %1;" ::"l"(addr), "h"(__bfloat16_as_ushort(__float2bfloat16_rn(v))) : "memory");
    }
}
// the value a plane of element type OT holds for the fp32 power v (what fdas_peaks will read back)
template <typename OT>
__device__ __forceinline__ float stored_value(float v)
{
    if constexpr (sizeof(OT) == 4) return v;
    else return __bfloat162float(__float2bfloat16_rn(v));
}

constexpr uint32_t TC_NO_ROW = 0xFFFFFFFFu;   // row-offset table: this |z| has no such plane row

// |.|^2 of Y_{+|z|} and Y_{-|z|} for the eight |z| of one 16-column chunk (file header) and the
// stores.  v[0..15] = (Ure_e, Ure_e+1, Vre_e, Vre_e+1) per entry pair, v[16..31] likewise for
// Uim, Vim, of this thread's output bin;
// o4[0..3] = row offsets (+|z|, -|z|) of two |z| each, in plane elements.
// FAST: the tile lies inside the plane and every entry has both rows -> straight-line code.
// Returns the largest power this thread stored (0 if none): the fused search flags the chunk
// when it exceeds the threshold (fdas_search).
template <bool FAST, typename OT>
__device__ __forceinline__ float epilogue_chunk(const uint32_t *v, const uint4 *o4, OT *out, bool ok)
{
    float mx = 0.f;
#pragma unroll
    for (int e2 = 0; e2 < 4; ++e2) {
        const uint4 o = o4[e2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const uint32_t offp = s ? o.z : o.x, offm = s ? o.w : o.y;
            const float ure = __uint_as_float(v[4 * e2 + s]), vre = __uint_as_float(v[4 * e2 + 2 + s]);
            const float uim = __uint_as_float(v[16 + 4 * e2 + s]), vim = __uint_as_float(v[16 + 4 * e2 + 2 + s]);
            if (FAST) {
                const float a = ure - vim, b = uim + vre, c = ure + vim, d = uim - vre;
                const float pp = __fmaf_rn(b, b, __fmul_rn(a, a)), pm = __fmaf_rn(d, d, __fmul_rn(c, c));   // as the bulk kernel
                st_cs_at(out, offp, pp);
                st_cs_at(out, offm, pm);
                mx = fmaxf(mx, fmaxf(pp, pm));
            } else {
                if (offp != TC_NO_ROW && ok) {
                    const float a = ure - vim, b = uim + vre;
                    const float pp = __fmaf_rn(b, b, __fmul_rn(a, a));
                    st_cs_at(out, offp, pp);
                    mx = fmaxf(mx, pp);
                }
                if (offm != TC_NO_ROW && ok) {
                    const float c = ure + vim, d = uim - vre;
                    const float pm = __fmaf_rn(d, d, __fmul_rn(c, c));
                    st_cs_at(out, offm, pm);
                    mx = fmaxf(mx, pm);
                }
            }
        }
    }
    return mx;
}

// fused search: "some power of bin r in the 8 |z| entries starting at table entry zi0 exceeds thr"
__device__ __noinline__ void flag_candidate(fdas_peak_t *cand, int *cand_count, int cand_capacity, int zi0, int r,
                                            float mx)
{
    const int slot = atomicAdd(cand_count, 1);
    if (slot < cand_capacity) {
        fdas_peak_t rec;
        rec.z_index = zi0;
        rec.r = r;
        rec.power = mx;
        cand[slot] = rec;
    }
}

// One tile for one epilogue warp: chunks HALF, HALF+2, ... of the NCH 16-column chunks.  The
// TMEM load of the next chunk is in flight while the current one is squared and stored, and
// the TMEM stage is handed back to the MMA issuer as soon as the last load has landed.
template <int NCH, int HALF, typename OT>
__device__ __forceinline__ void epilogue_tile(uint32_t taddr, const uint4 *otab4, OT *out, bool inside, bool ok,
                                              int full_chunks, uint32_t empty_bar, int lane,
                                              const fdas_search_args &sa, float thr, int zi_group0, long long col)
{
    constexpr int NMY = (NCH - HALF + 1) / 2;
    constexpr uint32_t NT = 16 * NCH;
    uint32_t v[2][32];
    if (NMY > 0) tmem_ld32(taddr + HALF * 16, taddr + NT + HALF * 16, v[0]);
#pragma unroll
    for (int i = 0; i < NMY; ++i) {
        const int c = HALF + 2 * i;
        tmem_ld_wait(v[i & 1]);
        if (i + 1 < NMY) tmem_ld32(taddr + (c + 2) * 16, taddr + NT + (c + 2) * 16, v[(i + 1) & 1]);
        if (i + 1 == NMY) {
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_bar);
        }
        float mx;
        if (inside && c < full_chunks) mx = epilogue_chunk<true, OT>(v[i & 1], otab4 + 4 * c, out, true);
        else mx = epilogue_chunk<false, OT>(v[i & 1], otab4 + 4 * c, out, ok);
        mx = stored_value<OT>(mx);   // rounding is monotone: the largest stored value
        if (mx > thr)   // thr = +inf unless fdas_search
            flag_candidate(sa.cand, sa.cand_count, sa.cand_capacity, zi_group0 + 8 * c, (int)col, mx);
    }
    if (NMY == 0) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar);
    }
}

// One lane of a converged warp (elect.sync), as a predicate value
__device__ __forceinline__ uint32_t elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred;
}
// umma_bf16 issued by the elected lane only; every lane of the warp executes the surrounding code,
// so the descriptors stay in uniform registers and MMAs issue back to back.  The descriptors come as their low
// words (the address field moves, 32-bit adds) and the constant high word TC_DESC_HI.
__device__ __forceinline__ void umma_bf16_elected(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t idesc,
                                                  uint32_t accumulate, uint32_t elected)
{
    asm volatile(
        "{\n\t.reg .pred p, q;\n\t.reg .b64 da, db;\n\t"
        "mov.b64 da, {%1, %6};\n\t"
        "mov.b64 db, {%2, %6};\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "setp.ne.b32 q, %5, 0;\n\t"
        "@q tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_lo), "r"(b_lo), "r"(idesc), "r"(accumulate), "r"(elected), "r"(TC_DESC_HI)
        : "memory");
}
__device__ __forceinline__ void umma_commit_elected(uint32_t bar, uint32_t elected)
{
    asm volatile(
        "{\n\t.reg .pred q;\n\t"
        "setp.ne.b32 q, %1, 0;\n\t"
        "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}"
        ::"r"(bar), "r"(elected)
        : "memory");
}

// The MMA warp of both kernels.  Per tile 2 KS MMAs (K steps outermost, so consecutive MMAs
// alternate between the re and im accumulators), then a commit that signals the epilogue.
//
// The tensor pipe queues only a few MMAs (measured with clock64 stamps: the issuing thread reaches the end of a
// tile when that tile is one or two MMAs from done), so whatever the thread does between the last MMA of one tile
// and the first of the next is idle tensor time (measured: ~100 cycles per tile, 400-550 per item boundary with the
// waits and the item arithmetic at the top of the loops).  Everything the next tile needs -- its TMEM stage handed
// back by the epilogue, across an item boundary also the next Z buffer, the next item's tile count, the next tile's
// descriptors -- is therefore waited for / worked out BEFORE the last K step of the current tile is issued, and the
// loop is flat: commit, a few register moves, next tile's first MMA.
template <int NT, int SPLIT = 1, int MODE = TB_PLANE>
__device__ __forceinline__ void mma_issuer(const TcParams &p, uint32_t s_base, uint32_t off_z, uint32_t z_buf_bytes,
                                           uint32_t z_part_bytes, uint32_t z_full, uint32_t z_empty, uint32_t t_full,
                                           uint32_t t_empty, uint32_t tmem_base, uint32_t n_items, TbCta cta)
{
    // K steps run in the same order in every launch (the sums must agree bit for bit between fdas_convolve and the
    // plane-free search): the full-width step holding tap 0 first -- it initialises every column -- then on through
    // the taps, wrapping round (p.steps[] lists them in that order, fdas_mma_plan).  p.trim: a step multiplies only the
    // columns whose templates reach it, i.e. uses the table's instruction descriptor (fdas_tc_trims decides per launch).
    // (uniform in the compiler's eyes, see below)
    const int grp = (int)__reduce_max_sync(0xffffffffu, (unsigned)cta.grp);
    const uint32_t cta_x = __reduce_max_sync(0xffffffffu, cta.x<MODE>(p)), cta_nx = __reduce_max_sync(0xffffffffu, cta.nx<MODE>(p));
    const int KSg = p.nsteps[grp < FDAS_TC_STEP_TABLES - 1 ? grp : FDAS_TC_STEP_TABLES - 1];   // K steps of this group
    const unsigned long long *const steps = p.steps[grp < FDAS_TC_STEP_TABLES - 1 ? grp : FDAS_TC_STEP_TABLES - 1];
    constexpr uint32_t b_lbo = (uint32_t)NT * 16u;   // next 8-tap chunk of the tap matrix
    const uint32_t elected = elect_one();
    const uint32_t b_lo0 = smem_desc_lo(s_base, b_lbo);
    // SPLIT == 3 (fp32 variant): x = x1 + x2, h = h1 + h2 in bf16 terms; x h ~ x1 h1 + x1 h2 + x2 h1
    // (the dropped x2 h2 is <= 2^-18 |x h|).  Z parts: re1, im1, re2, im2; tap images: h1, h2.
    const uint32_t b2_off = (2u * (uint32_t)p.KS * b_lbo) >> 4;   // second tap-matrix image
    const uint32_t a2_off = (2u * z_part_bytes) >> 4;             // re2 / im2 parts
    // One K step of one tile; descriptors advance by adding to their 14-bit address field (units of 16 bytes;
    // shared memory is < 256 KB, so no carry leaves the field).
    auto issue_step = [&](uint32_t d_re, uint32_t d_im, uint32_t a_re, uint32_t a_im, int i, uint32_t acc) {
        const unsigned long long e = steps[i];
        const uint32_t idesc = p.trim ? (uint32_t)e : tc_idesc((uint32_t)NT);
        const uint32_t a_off = (uint32_t)(e >> 32) & 0xFFFFu, b_off = (uint32_t)(e >> 48);
        const uint32_t ar = a_re + a_off, ai = a_im + a_off, bk = b_lo0 + b_off;
        umma_bf16_elected(d_re, ar, bk, idesc, acc, elected);
        umma_bf16_elected(d_im, ai, bk, idesc, acc, elected);
        if constexpr (SPLIT == 3) {
            umma_bf16_elected(d_re, ar, bk + b2_off, idesc, 1, elected);
            umma_bf16_elected(d_im, ai, bk + b2_off, idesc, 1, elected);
            umma_bf16_elected(d_re, ar + a2_off, bk, idesc, 1, elected);
            umma_bf16_elected(d_im, ai + a2_off, bk, idesc, 1, elected);
        }
    };
    // TB_RECHECK: the items are separated by barriers the loader and (clustered) this warp take part in, so nothing
    // of the next item is waited for early there
    constexpr bool AHEAD_ITEM = MODE != TB_RECHECK;
    if (cta_x >= n_items) return;
    // Tiles of an item.  Everything the issue loop branches on must be warp-uniform IN THE COMPILER'S EYES: the
    // descriptors live in uniform registers, and one branch on a value held in a vector register drags every
    // loop-carried descriptor into vector registers at the price of a R2UR per MMA operand (measured: 1120 -> 1360
    // cycles per tile).  The tile counts therefore pass through a warp reduction (REDUX writes a uniform register);
    // the block index inside the series is tracked by subtraction instead of it % n_blocks (no division between MMAs).
    n_items = __reduce_max_sync(0xffffffffu, n_items);
    uint32_t blk_cur = cta_x;
    auto blk_wrap = [&](uint32_t b) {
        while (b >= (uint32_t)p.n_blocks) b -= (uint32_t)p.n_blocks;
        return b;
    };
    auto tiles_of = [&](uint32_t item, uint32_t blk) {
        if constexpr (MODE == TB_RECHECK) {
            long long ser_, blk0_;
            int nt, centre_;
            tb_item<MODE>(p, item, ser_, blk0_, nt, centre_);
            return (int)__reduce_max_sync(0xffffffffu, (unsigned)nt);
        } else {
            const long long left = p.M - (long long)(p.blk_first + blk) * p.R;
            return (int)__reduce_max_sync(0xffffffffu, (unsigned)(((left < p.R ? left : (long long)p.R) + 128 - 1) >> 7));
        }
    };
    blk_cur = blk_wrap(blk_cur);
    auto wait_stage = [&](uint32_t tt) { mbar_wait(t_empty + 8 * (tt & 1), ((tt >> 1) & 1) ^ 1); };
    auto wait_z = [&](uint32_t nn) { mbar_wait(z_full + 8 * (nn & 1), (nn >> 1) & 1); };
    // the tile being issued: item `it` (the n-th of this CTA, `n_tiles` tiles), tile `tile` of it, the t-th tile overall
    uint32_t it = cta_x, n = 0, t = 0;
    int tile = 0, n_tiles = tiles_of(it, blk_cur), n_tiles_next = 0;
    uint32_t z_addr = s_base + off_z;
    wait_z(0);
    wait_stage(0);
    tc_fence_after();
    uint32_t d_re = tmem_base;
    uint32_t a_re = smem_desc_lo(z_addr, 128u), a_im = smem_desc_lo(z_addr + z_part_bytes, 128u);
    for (;;) {
        const uint32_t stage = t & 1;
        issue_step(d_re, d_re + NT, a_re, a_im, 0, 0);
        // the next item's tile count, early in the current item
        const bool has_next = it + cta_nx < n_items;
        if (tile == 0 && has_next) {
            blk_cur = blk_wrap(blk_cur + cta_nx);
            n_tiles_next = tiles_of(it + cta_nx, blk_cur);
        }
#pragma unroll 2
        for (int i = 1; i + 1 < KSg; ++i) issue_step(d_re, d_re + NT, a_re, a_im, i, 1);
        // ---- ahead of the last K step: the next tile's operands, and what it waits for
        const bool item_ends = tile + 1 == n_tiles;
        bool more = true, late_waits = false;
        uint32_t nz_addr = z_addr;
        if (!item_ends) {
            wait_stage(t + 1);
        } else if (!has_next) {
            more = false;
        } else {
            nz_addr = s_base + off_z + ((n + 1) & 1) * z_buf_bytes;
            if (AHEAD_ITEM) {
                wait_z(n + 1);
                wait_stage(t + 1);
            } else {
                late_waits = true;
            }
        }
        const int ntile = item_ends ? 0 : tile + 1;
        const uint32_t nd_re = tmem_base + ((t + 1) & 1) * TC_STAGE_COLS;
        const uint32_t na_re = smem_desc_lo(nz_addr + (uint32_t)(ntile * TC_TILE) * 16u, 128u);
        const uint32_t na_im = smem_desc_lo(nz_addr + z_part_bytes + (uint32_t)(ntile * TC_TILE) * 16u, 128u);
        if (KSg > 1) issue_step(d_re, d_re + NT, a_re, a_im, KSg - 1, 1);
        umma_commit_elected(t_full + 8 * stage, elected);
        if (item_ends) {
            umma_commit_elected(z_empty + 8 * (n & 1), elected);
            if constexpr (MODE == TB_RECHECK) {
                if (p.clustered) {   // a cluster barrier counts every thread (see tb_item_sync)
                    tb_item_sync(1, 0);
                    tb_item_sync(1, 0);
                }
            }
            if (!more) break;
            it += cta_nx;
            n += 1;
            n_tiles = n_tiles_next;
        }
        ++t;
        tile = ntile;
        z_addr = nz_addr;
        d_re = nd_re;
        a_re = na_re;
        a_im = na_im;
        if (late_waits) {
            wait_z(n);
            wait_stage(t);
        }
        tc_fence_after();
    }
}

// The loader warps of both kernels: per work item, the spectrum block -> bf16 (round to nearest
// even, reading A12) -> the Z rows (file header) of buffer n & 1.  The global loads of
// item n+1 are issued before the wait for buffer n and stay in registers across it, so that
// their latency hides behind the tensor core working on the previous items.
constexpr int TC_LD_ITERS = 8;   // sample pairs per loader thread: (R + 16 KS) / 2 / 96 <= (1024 + 512) / 192
constexpr int TC_LD_PAIRS = 2;   // Z row pairs a loader thread has in flight (phase B of spectrum_loader)

template <int MODE = TB_PLANE>
__device__ __forceinline__ void loader_fetch(const TcParams &p, uint32_t it, uint32_t xn, int lt, float2 (&a)[TC_LD_ITERS],
                                             float2 (&b)[TC_LD_ITERS])
{
    long long ser, blk0;
    int n_tiles_, centre_;
    tb_item<MODE>(p, it, ser, blk0, n_tiles_, centre_);
    const long long g0 = blk0 - p.M0;   // sample index of xs[0]
    const float2 *__restrict__ X = p.spectra + (size_t)ser * p.M;
#pragma unroll
    for (int i = 0; i < TC_LD_ITERS; ++i) {
        const uint32_t pi = lt + i * TC_LOAD_THREADS;
        const long long g = g0 + 2 * (long long)pi;
        a[i] = make_float2(0.f, 0.f);
        b[i] = make_float2(0.f, 0.f);
        if (pi < xn / 2) {
            if (g >= 0 && g < p.M) a[i] = __ldg(X + g);
            if (g + 1 >= 0 && g + 1 < p.M) b[i] = __ldg(X + g + 1);
        }
    }
}

// residual of the bf16 rounding: x - bf16(x) is exact in fp32 (x has 24 significant bits, bf16(x) the top 8)
__device__ __forceinline__ float bf16_residual(float x) { return x - __bfloat162float(__float2bfloat16_rn(x)); }

template <int SPLIT = 1, int MODE = TB_PLANE>
__device__ __forceinline__ void spectrum_loader(const TcParams &p, unsigned char *smem, uint32_t off_xs,
                                                uint32_t xs_part_bytes, uint32_t xn, uint32_t off_z, uint32_t z_buf_bytes,
                                                uint32_t z_part_bytes, uint32_t zr, uint32_t z_full, uint32_t z_empty,
                                                int lt, uint32_t n_items, TbCta cta, float2 (&a)[TC_LD_ITERS], float2 (&b)[TC_LD_ITERS])
{
    // sample planes: re, im of the bf16 spectrum; SPLIT == 3 adds re, im of the rounded residual (parts 2, 3)
    constexpr int NP = SPLIT == 3 ? 4 : 2;
    uint32_t *xs_re = reinterpret_cast<uint32_t *>(smem + off_xs);
    uint32_t *xs_im = reinterpret_cast<uint32_t *>(smem + off_xs + xs_part_bytes);
    uint32_t n = 0;   // a, b: the first item's samples, fetched by the kernel before its set-up (tb_first_fetch)
    for (uint32_t it = cta.x<MODE>(p); it < n_items; it += cta.nx<MODE>(p), ++n) {
        const uint32_t buf = n & 1, zuse = n >> 1;
        // phase A: spectrum block -> bf16 (round-to-nearest-even), re and im planes
#pragma unroll
        for (int i = 0; i < TC_LD_ITERS; ++i) {
            const uint32_t pi = lt + i * TC_LOAD_THREADS;
            if (pi < xn / 2) {
                xs_re[pi] = pack_bf16(a[i].x, b[i].x);
                xs_im[pi] = pack_bf16(a[i].y, b[i].y);
                if (SPLIT == 3) {
                    xs_re[pi + xs_part_bytes / 2] = pack_bf16(bf16_residual(a[i].x), bf16_residual(b[i].x));
                    xs_im[pi + xs_part_bytes / 2] = pack_bf16(bf16_residual(a[i].y), bf16_residual(b[i].y));
                }
            }
        }
        named_bar_sync(1, TC_LOAD_THREADS);
        if (it + cta.nx<MODE>(p) < n_items) loader_fetch<MODE>(p, it + cta.nx<MODE>(p), xn, lt, a, b);
        mbar_wait<64>(z_empty + 8 * buf, (zuse & 1) ^ 1);
        // phase B: Z row i = samples i .. i+7 (16 bytes), for every part.  A thread builds the row pair (2q, 2q+1)
        // from the five words xs[q .. q+4] (the odd row is the even one shifted by one sample); the loads of TC_LD_PAIRS
        // pairs and all parts are issued before the first store: the tensor core's operand reads keep shared memory
        // ~90 % busy, a dependent load -> store chain per row took the loader a whole item period (measured), which
        // left the MMA warp waiting at every item boundary.  Lanes with bit 2 set store their odd row first: the
        // eight lanes of a quarter warp then cover 32 distinct banks (rows 2q of lanes 0-3, rows 2q+1 of lanes 4-7).
        unsigned char *zb = smem + off_z + buf * z_buf_bytes;
        const uint32_t n_pairs = zr >> 1;   // zr = R + 16 KS - 8 is even
        const bool odd_first = (lt & 4) != 0;
        for (uint32_t q0 = lt; q0 < n_pairs; q0 += TC_LD_PAIRS * TC_LOAD_THREADS) {
            uint32_t w[TC_LD_PAIRS][NP][5];
#pragma unroll
            for (int u = 0; u < TC_LD_PAIRS; ++u) {
                const uint32_t q = q0 + u * TC_LOAD_THREADS;
                if (q < n_pairs) {
#pragma unroll
                    for (int part = 0; part < NP; ++part) {
                        const uint32_t *src = xs_re + part * (xs_part_bytes / 4) + q;
#pragma unroll
                        for (int j = 0; j < 5; ++j) w[u][part][j] = src[j];
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < TC_LD_PAIRS; ++u) {
                const uint32_t q = q0 + u * TC_LOAD_THREADS;
                if (q < n_pairs) {
#pragma unroll
                    for (int part = 0; part < NP; ++part) {
                        const uint32_t *v = w[u][part];
                        const uint4 even = make_uint4(v[0], v[1], v[2], v[3]);
                        const uint4 odd = make_uint4(__byte_perm(v[0], v[1], 0x5432), __byte_perm(v[1], v[2], 0x5432),
                                                     __byte_perm(v[2], v[3], 0x5432), __byte_perm(v[3], v[4], 0x5432));
                        uint4 *rows = reinterpret_cast<uint4 *>(zb + part * z_part_bytes) + 2 * (size_t)q;
                        rows[odd_first ? 1 : 0] = odd_first ? odd : even;
                        rows[odd_first ? 0 : 1] = odd_first ? even : odd;
                    }
                }
            }
        }
        fence_proxy_async();   // generic-proxy writes of Z -> visible to tcgen05.mma
        mbar_arrive(z_full + 8 * buf);
        named_bar_sync(1, TC_LOAD_THREADS);   // xs is rewritten by the next item
        if constexpr (MODE == TB_RECHECK) {
            if (p.clustered) {
                tb_item_sync(1, 0);
                tb_item_sync(1, 0);
            }
        }
    }
}

template <int NCH, typename OT>
__global__ void __launch_bounds__(TC_THREADS, 1) fdas_mma_convolve_kernel(const TcParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NT = 16 * NCH;
    const TcSmem L(p.R, p.KS, NT);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const TbCta cta = tb_cta<TB_PLANE>(p);
    const int grp = cta.grp;
    const uint32_t n_items = (uint32_t)p.batch * (uint32_t)p.n_blocks;

    const uint32_t s_base = smem_u32(smem);
    const uint32_t bars = s_base + L.off_bars;
    // barrier slots: z_full[2] (loader -> mma), z_empty[2] (mma -> loader),
    //                t_full[2] (mma -> epilogue), t_empty[2] (epilogue -> mma)
    const uint32_t z_full = bars, z_empty = bars + 16, t_full = bars + 32, t_empty = bars + 48;
    uint32_t *holder = reinterpret_cast<uint32_t *>(smem + L.off_holder);
    uint2 *otab = reinterpret_cast<uint2 *>(smem + L.off_ktab);   // [NT/2] row offsets (+|z|, -|z|)

    // the loader warps put the global loads of their first item in flight before the set-up: its latency hides behind
    // the tap-matrix copy and the TMEM allocation (a launch of config 1 is 10 us long, the set-up 3 of them)
    float2 first_a[TC_LD_ITERS], first_b[TC_LD_ITERS];
    if (warp >= TC_LOAD_WARP0 && cta.x<TB_PLANE>(p) < n_items)
        loader_fetch<TB_PLANE>(p, cta.x<TB_PLANE>(p), L.xn, threadIdx.x - TC_LOAD_WARP0 * 32, first_a, first_b);
    // ---- one-time setup: tap matrix image and row-offset table -> shared memory, barriers, TMEM
    {
        const uint4 *src = p.bmat + (size_t)grp * (L.b_bytes / 16);
        uint4 *dst = reinterpret_cast<uint4 *>(smem);
        for (uint32_t i = threadIdx.x; i < L.b_bytes / 16; i += TC_THREADS) dst[i] = __ldg(src + i);
        for (int i = threadIdx.x; i < NT / 2; i += TC_THREADS) {
            int2 kk = make_int2(-1, -1);
            if (i < p.nzg) kk = p.ktab[(size_t)grp * p.nzg + i];
            otab[i] = make_uint2(kk.x >= 0 ? (uint32_t)((long long)kk.x * p.M) : TC_NO_ROW,
                                 kk.y >= 0 ? (uint32_t)((long long)kk.y * p.M) : TC_NO_ROW);
        }
        fence_proxy_async();   // the tap matrix is read by the tensor core (async proxy)
    }
    if (threadIdx.x == 0 && blockIdx.x == 0 && p.search.enabled) {
        *p.search.cand_count_next = 0;   // the other counter: nobody appends to it during this launch
        *p.search.count_out = 0;         // written by the resolve kernel that follows in stream order
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(z_full + 8 * s, TC_LOAD_THREADS);
            mbar_init(z_empty + 8 * s, 1);
            mbar_init(t_full + 8 * s, 1);
            mbar_init(t_empty + 8 * s, TC_EPI_WARPS);
        }
        fence_barrier_init();
    }
    if (warp == TC_MMA_WARP) tmem_alloc(smem_u32(holder), TC_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *holder;

    if (warp < TC_EPI_WARPS) {
        // =========================== epilogue ===========================
        const int q = warp & 3, half = warp >> 2;
        const uint4 *otab4 = reinterpret_cast<const uint4 *>(otab);
        const float thr = p.search.enabled ? p.search.thr : __int_as_float(0x7f800000);
        const int zi_group0 = grp * p.nzg;
        uint32_t t = 0;
        for (uint32_t it = cta.x<TB_PLANE>(p); it < n_items; it += cta.nx<TB_PLANE>(p)) {
            const long long ser = it / (uint32_t)p.n_blocks;   // 32-bit division: items < 2^31 (checked by the launcher)
            const long long blk0 = (long long)(it % (uint32_t)p.n_blocks) * p.R;
            const long long left = p.M - blk0;
            const int n_tiles = (int)((left < p.R ? left : p.R) + TC_TILE - 1) / TC_TILE;
            for (int tile = 0; tile < n_tiles; ++tile, ++t) {
                const uint32_t stage = t & 1, use = t >> 1;
                const long long col0 = blk0 + tile * TC_TILE;
                const long long col = col0 + q * 32 + lane;
                OT *const out = static_cast<OT *>(p.planes) + (size_t)ser * p.K * p.M + col;
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + stage * TC_STAGE_COLS;
                const bool inside = col0 + TC_TILE <= p.M;
                mbar_wait(t_full + 8 * stage, use & 1);
                tc_fence_after();
                if (half == 0)
                    epilogue_tile<NCH, 0, OT>(taddr, otab4, out, inside, col < p.M, p.full_chunks, t_empty + 8 * stage, lane,
                                          p.search, thr, zi_group0, col);
                else
                    epilogue_tile<NCH, 1, OT>(taddr, otab4, out, inside, col < p.M, p.full_chunks, t_empty + 8 * stage, lane,
                                          p.search, thr, zi_group0, col);
            }
        }
    } else if (warp == TC_MMA_WARP) {
        // =========================== MMA issuer ===========================
        mma_issuer<NT, 1, TB_PLANE>(p, s_base, L.off_z, L.z_buf_bytes, L.z_part_bytes, z_full, z_empty, t_full, t_empty,
                                    __shfl_sync(0xffffffffu, tmem_base, 0), n_items, cta);
    } else {
        // =========================== loader ===========================
        spectrum_loader(p, smem, L.off_xs, L.xs_part_bytes, L.xn, L.off_z, L.z_buf_bytes, L.z_part_bytes, L.zr, z_full,
                        z_empty, threadIdx.x - TC_LOAD_WARP0 * 32, n_items, cta, first_a, first_b);
    }

    tc_fence_before();
    __syncthreads();
    if (warp == TC_MMA_WARP) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc(tmem_base, TC_TMEM_COLS);
    }
}

// =====================================================================================
// fdas_mma_bulk_kernel: the same loader and MMA issuer; the epilogue stages the powers in
// shared memory and writes the plane with bulk copies.
// =====================================================================================
// warp roles: 8 SETS epilogue warps (4 TMEM lane quarters x 2 halves per set), then the MMA warp, then the loader
__host__ __device__ constexpr int tb_sets(int split) { return split == 3 ? 1 : 2; }
__host__ __device__ constexpr int tb_epi_warps(int split) { return 8 * tb_sets(split); }
__host__ __device__ constexpr int tb_threads(int split) { return 32 * (tb_epi_warps(split) + 1 + TC_LOAD_WARPS); }   // 640 / 384
constexpr int TB_CGROUPS = 4;           // column groups: NCH entry pairs (4 NCH columns per part) each
// Recheck launch with one template group: the powers of the listed tile go to a strip in shared memory, K rows of
// (last bin of the left neighbour tile | the 128 bins of the tile | first bin of the right neighbour tile), padded
constexpr int TB_STRIP_W = 132;
constexpr int TB_BOXES = FDAS_TC_MAX_BOXES;   // tensor maps, one per distinct run length (plan->tc_box_heights)
struct TbMaps {
    CUtensorMap m[TB_BOXES];            // the planes as a [batch*K][M] fp32 matrix, box = tc_box_heights[i] rows x 128 bins
};

// shared-memory carve-up of the bulk kernel.  ROWB = bytes of one staging row (one plane row
// segment pushed out by one bulk copy): 128 bins x 4 B.
struct TbSmem {
    uint32_t b_bytes, zr, z_part_bytes, z_buf_bytes, xn, xs_part_bytes, slots, stage_cg_bytes;
    uint32_t off_z, off_xs, off_stage, off_bars, off_holder, total;
    // split = 1: bf16 operands; split = 3: the fp32 variant, every operand split into two bf16 terms
    // (two tap-matrix images, four Z parts) and one epilogue warp set (one staging buffer per column group)
    // staging: the box-store staging rows; strip_rows > 0 (recheck launch, one template group): no staging, a strip
    // of strip_rows x TB_STRIP_W floats in its place
    __host__ __device__ TbSmem(int R, int KS, int NT, int rowb, int split, bool staging = true, int strip_rows = 0)
    {
        const uint32_t TP = 16u * KS;
        const uint32_t nb = split == 3 ? 2u : 1u, np = 2u * nb, sets = split == 3 ? 1u : 2u;
        b_bytes = 2u * KS * NT * 16u;               // one tap-matrix image
        zr = R + TP - 8;
        z_part_bytes = zr * 16u;
        z_buf_bytes = np * z_part_bytes;
        xn = R + TP;
        xs_part_bytes = xn * 2u;
        slots = (uint32_t)NT / 4u;                 // 4 NCH
        stage_cg_bytes = slots * (uint32_t)rowb;   // one buffer of one column group
        off_z = nb * b_bytes;
        off_xs = off_z + 2u * z_buf_bytes;
        off_stage = (off_xs + np * xs_part_bytes + 127u) & ~127u;
        off_bars = (off_stage + (strip_rows > 0 ? (uint32_t)strip_rows * TB_STRIP_W * 4u : staging ? sets * TB_CGROUPS * stage_cg_bytes : 0u) + 15u) & ~15u;
        off_holder = off_bars + 8u * 8u;
        total = off_holder + 16u;
    }
};

// TMEM -> registers, this warp's 32 lanes x N consecutive columns (N a multiple of 4, <= 32)
template <int N>
__device__ __forceinline__ void tmem_ld_cols(uint32_t taddr, uint32_t *v)
{
    if constexpr (N >= 16) {
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
              "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
            : "r"(taddr)
            : "memory");
        tmem_ld_cols<N - 16>(taddr + 16, v + 16);
    } else if constexpr (N >= 8) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                     : "r"(taddr)
                     : "memory");
        tmem_ld_cols<N - 8>(taddr + 8, v + 8);
    } else if constexpr (N >= 4) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3])
                     : "r"(taddr)
                     : "memory");
        tmem_ld_cols<N - 4>(taddr + 4, v + 4);
    }
}
// tcgen05.wait::ld, then pin every loaded register behind it (an empty asm the compiler cannot
// hoist a use across)
template <int N>
__device__ __forceinline__ void tmem_ld_fence(uint32_t *v)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < N; ++i) asm volatile("" : "+r"(v[i]));
}

// packed fp32x2 arithmetic (FADD2 / FMUL2 / FFMA2 on sm_100a)
__device__ __forceinline__ unsigned long long f2_pack(uint32_t lo, uint32_t hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ void f2_unpack(unsigned long long v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long f2_add(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long f2_sub(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// smem box [h][128] floats (dense rows) -> plane rows row..row+h-1, bins col..col+127 (clipped at M)
__device__ __forceinline__ void tensor_store(const CUtensorMap *map, uint32_t ssrc, int col, int row)
{
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(map), "r"(col),
                 "r"(row), "r"(ssrc)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

template <int NCH, typename OT, int SPLIT, int MODE = TB_PLANE>
__global__ void __launch_bounds__(tb_threads(SPLIT), 1)
fdas_mma_bulk_kernel(const TcParams p, const __grid_constant__ TbMaps maps)
{
    static_assert(MODE == TB_PLANE || sizeof(OT) == 4, "plane-free search computes float powers");
    constexpr int SETS = tb_sets(SPLIT), TB_EPI_WARPS = tb_epi_warps(SPLIT), TB_MMA_WARP = TB_EPI_WARPS,
                  TB_LOAD_WARP0 = TB_EPI_WARPS + 1, TB_THREADS = tb_threads(SPLIT);
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NT = 16 * NCH;
    constexpr int NC = 4 * NCH;            // columns per part per column group = staging rows (slots)
    constexpr uint32_t ROWB = TC_TILE * sizeof(OT);   // bytes of one staging row
    // recheck launch of a single template group: the strip lives in shared memory (no scratch round trip through L2)
    const bool smem_strip = MODE == TB_RECHECK && gridDim.y == 1;
    const TbCta cta = tb_cta<MODE>(p);
    const TbSmem L(p.R, p.KS, NT, ROWB, SPLIT, MODE != TB_SCAN, smem_strip ? p.K : 0);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = cta.grp;
    if (MODE == TB_RECHECK) asm volatile("griddepcontrol.wait;" ::: "memory");   // the scan launch has listed its tiles
    const uint32_t n_items = tb_items<MODE>(p);
    if (MODE == TB_RECHECK && blockIdx.x >= n_items) return;   // nothing flagged for this CTA (its whole cluster: same x)

    const uint32_t s_base = smem_u32(smem);
    const uint32_t bars = s_base + L.off_bars;
    const uint32_t z_full = bars, z_empty = bars + 16, t_full = bars + 32, t_empty = bars + 48;
    uint32_t *holder = reinterpret_cast<uint32_t *>(smem + L.off_holder);

    // the loader warps put the global loads of their first item in flight before the set-up (see fdas_mma_convolve_kernel)
    float2 first_a[TC_LD_ITERS], first_b[TC_LD_ITERS];
    if (warp >= TB_LOAD_WARP0 && cta.x<MODE>(p) < n_items)
        loader_fetch<MODE>(p, cta.x<MODE>(p), L.xn, threadIdx.x - TB_LOAD_WARP0 * 32, first_a, first_b);
    // ---- one-time setup: tap matrix image -> shared memory, barriers, TMEM
    {
        // tap-matrix image(s) of this template group: bmat is [image][group][...]
        uint4 *dst = reinterpret_cast<uint4 *>(smem);
        for (int img = 0; img < (SPLIT == 3 ? 2 : 1); ++img) {
            const uint4 *src = p.bmat + ((size_t)img * p.groups + grp) * (L.b_bytes / 16);
            for (uint32_t i = threadIdx.x; i < L.b_bytes / 16; i += TB_THREADS) dst[img * (L.b_bytes / 16) + i] = __ldg(src + i);
        }
        fence_proxy_async();
    }
    if (MODE == TB_PLANE && threadIdx.x == 0 && blockIdx.x == 0 && p.search.enabled) {
        *p.search.cand_count_next = 0;
        *p.search.count_out = 0;
    }
    if (MODE == TB_SCAN && blockIdx.x == 0) {
        if (threadIdx.x == 0) *p.search.tile_count_next = 0;
        for (int i = threadIdx.x; i < p.batch; i += TB_THREADS) p.search.counts[i] = 0;
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < 2; ++s) {
            mbar_init(z_full + 8 * s, TC_LOAD_THREADS);
            mbar_init(z_empty + 8 * s, 1);
            mbar_init(t_full + 8 * s, 1);
            mbar_init(t_empty + 8 * s, 8);   // the eight epilogue warps that read stage s
        }
        fence_barrier_init();
    }
    if (warp == TB_MMA_WARP) tmem_alloc(smem_u32(holder), TC_TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *holder;

    if (warp < TB_EPI_WARPS) {
        // =========================== epilogue ===========================
        // Two warp sets take alternate tiles (set = TMEM stage), so that one set's chain
        // TMEM load -> powers -> staging -> fence -> barrier -> store issue overlaps the other's.
        // Inside a set, warp (q, half) owns TMEM lane quarter q and column groups 2 half, 2 half + 1.
        const int q = warp & 3, half = (warp >> 2) & 1, set = warp >> 3;   // SETS == 1: set = 0 takes every tile
        const int lt = q * 32 + lane;                       // bin inside the tile = TMEM lane
        const float thr = p.search.enabled ? p.search.thr : __int_as_float(0x7f800000);
        // Staging rows of a column group (NC = 4 NCH rows of 128 bins): the -|z| rows of its entries
        // el = 0, 1, .. in rows el, the +|z| rows in rows NC-1-el, so that each block is a run of
        // consecutive plane rows in ascending order (ranges[]: row0_n, cnt_n / row0_p, cnt_p) and
        // leaves as ONE tensor-map box (ranges[]: the run length selects a map whose box has exactly
        // that many rows).  Two of the four warps sharing a staging block issue one box each: a
        // UTMASTG costs its issuing warp ~220 cycles (measured), which must not serialise.
        const bool issuer = q < 2 && lane == 0;
        const int bar_id = 2 + 2 * set + half;              // the 128 threads (set, half)
        // the row runs of this warp's two column groups, read once: nothing inside the tile loop may touch
        // global memory (a load behind the saturated write stream stalls its warp, and with it the barrier
        // of its staging block, for thousands of cycles)
        const int4 rg2[2] = {p.ranges[grp * TB_CGROUPS + 2 * half], p.ranges[grp * TB_CGROUPS + 2 * half + 1]};
        uint32_t t = 0;
        for (uint32_t it = cta.x<MODE>(p); it < n_items; it += cta.nx<MODE>(p)) {
            long long ser, blk0;
            int n_tiles, centre;
            tb_item<MODE>(p, it, ser, blk0, n_tiles, centre);
            for (int tile = 0; tile < n_tiles; ++tile, ++t) {
                if (SETS == 2 && (int)(t & 1) != set) continue;
                const uint32_t stage = t & 1, use = t >> 1;
                const uint32_t sblk = SETS == 2 ? stage : 0;   // staging buffer of this tile (per column group)
                const long long col0 = blk0 + tile * TC_TILE;
                const uint32_t taddr0 = tmem_base + ((uint32_t)(q * 32) << 16) + stage * TC_STAGE_COLS;
                mbar_wait(t_full + 8 * stage, use & 1);
                tc_fence_after();
                // ---- TMEM -> powers in registers, for both column groups, then hand the stage back at once:
                // the MMA of tile t+2 never waits for the store path (shared-memory staging, TMA backlog)
                float pw[2][NC];   // per column group: (pm0, pm1, pp0, pp1) of each entry pair
                float mx2[2];
#pragma unroll
                for (int pass = 0; pass < 2; ++pass) {
                    const int cg = 2 * half + pass;
                    float mx = 0.f;
#pragma unroll
                    for (int pr0 = 0; pr0 < NCH; pr0 += 4) {
                        constexpr int dummy = 0;
                        (void)dummy;
                        const int npr = NCH - pr0 < 4 ? NCH - pr0 : 4;   // entry pairs in this chunk (compile time after unrolling)
                        uint32_t v[32];
                        if (npr == 4) {
                            tmem_ld_cols<16>(taddr0 + cg * NC + 4 * pr0, v);
                            tmem_ld_cols<16>(taddr0 + NT + cg * NC + 4 * pr0, v + 16);
                        } else if (npr == 3) {
                            tmem_ld_cols<12>(taddr0 + cg * NC + 4 * pr0, v);
                            tmem_ld_cols<12>(taddr0 + NT + cg * NC + 4 * pr0, v + 16);
                        } else if (npr == 2) {
                            tmem_ld_cols<8>(taddr0 + cg * NC + 4 * pr0, v);
                            tmem_ld_cols<8>(taddr0 + NT + cg * NC + 4 * pr0, v + 16);
                        } else {
                            tmem_ld_cols<4>(taddr0 + cg * NC + 4 * pr0, v);
                            tmem_ld_cols<4>(taddr0 + NT + cg * NC + 4 * pr0, v + 16);
                        }
                        tmem_ld_fence<32>(v);
                        if (pass == 1 && pr0 + 4 >= NCH) {           // last load of this tile has landed
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(t_empty + 8 * stage);
                        }
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            if (i >= npr) continue;
                            const int pr = pr0 + i;
                            const unsigned long long ure = f2_pack(v[4 * i], v[4 * i + 1]), vre = f2_pack(v[4 * i + 2], v[4 * i + 3]);
                            const unsigned long long uim = f2_pack(v[16 + 4 * i], v[16 + 4 * i + 1]);
                            const unsigned long long vim = f2_pack(v[16 + 4 * i + 2], v[16 + 4 * i + 3]);
                            const unsigned long long a = f2_sub(ure, vim), b = f2_add(uim, vre);
                            const unsigned long long c = f2_add(ure, vim), d = f2_sub(uim, vre);
                            const unsigned long long pp = f2_fma(b, b, f2_mul(a, a)), pm = f2_fma(d, d, f2_mul(c, c));
                            f2_unpack(pm, pw[pass][4 * pr], pw[pass][4 * pr + 1]);
                            f2_unpack(pp, pw[pass][4 * pr + 2], pw[pass][4 * pr + 3]);
                            // padded columns give exactly zero; a sign whose row is not in the plane (asymmetric
                            // grids) can only add a candidate, which the resolve kernel then rejects
                            mx = fmaxf(mx, fmaxf(fmaxf(pw[pass][4 * pr], pw[pass][4 * pr + 1]),
                                                 fmaxf(pw[pass][4 * pr + 2], pw[pass][4 * pr + 3])));
                        }
                    }
                    mx2[pass] = stored_value<OT>(mx);   // rounding is monotone: the largest stored value
                }
                if constexpr (MODE == TB_SCAN) {
                    // plane-free search, first launch: nothing is stored.  A tile with a power above the threshold is
                    // listed once; bits 1 / 2 ask the recheck launch for the left / right neighbour tile as well
                    // (the 8-neighbourhood of a candidate in the first / last bin reaches into it).  Padded columns
                    // give exactly zero; a row that is not in the plane can only list a tile needlessly.
                    const bool hit = fmaxf(mx2[0], mx2[1]) > thr && col0 + lt < p.M;
                    const unsigned ball = __ballot_sync(0xffffffffu, hit);
                    if (ball != 0u && lane == 0) {
                        const int bits = 1 | ((q == 0 && (ball & 1u)) ? 2 : 0) | ((q == 3 && (ball >> 31)) ? 4 : 0);
                        const int tg = (int)(ser * p.tiles_per_series + (col0 >> 7));
                        if (atomicOr(p.search.tile_flags + tg, bits) == 0)
                            p.search.tile_list[atomicAdd(p.search.tile_count, 1)] = tg;
                    }
                    continue;
                }
                // bf16-stored plane: the powers go straight from registers to the plane (one 64-byte row segment per
                // warp and store).  Measured on config 3: 0.291 ms against 0.317 ms through staging + box stores (the
                // 16-bit staging stores cost more shared-memory time than the halved bytes save); for the float plane
                // the staged path wins (0.300 ms against 0.364 ms with direct stores).
                auto direct_pass = [&](int pass) {
                    const int cg = 2 * half + pass;
                    const int4 rg = rg2[pass];
                    const int cnt_n = rg.y & 0xFFFF, cnt_p = rg.w & 0xFFFF;
                    if (col0 + lt < p.M) {
                        OT *const out = static_cast<OT *>(p.planes) + (size_t)ser * p.K * p.M + col0 + lt;
                        const uint32_t Mu = (uint32_t)p.M;
                        if (cnt_n == 2 * NCH && cnt_p == 2 * NCH) {
                            // full column group: straight-line code, row offsets by addition
                            // two running row pointers, each advanced by one IMAD.WIDE (ptr += +-M * sizeof(OT))
                            long long pn, pp;
                            asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pn) : "r"((uint32_t)rg.x * Mu), "n"((int)sizeof(OT)), "l"(out));
                            asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pp) : "r"((uint32_t)(rg.z + cnt_p - 1) * Mu), "n"((int)sizeof(OT)), "l"(out));
                            const int Mi = (int)Mu;
#pragma unroll
                            for (int el = 0; el < 2 * NCH; ++el) {
                                const float vn = pw[pass][4 * (el >> 1) + (el & 1)], vp = pw[pass][4 * (el >> 1) + 2 + (el & 1)];
                                if constexpr (sizeof(OT) == 2) {
                                    asm volatile("st.global.cs.u16 [%0], %1;" ::"l"(pn), "h"(__bfloat16_as_ushort(__float2bfloat16_rn(vn))) : "memory");
                                    asm volatile("st.global.cs.u16 [%0], %1;" ::"l"(pp), "h"(__bfloat16_as_ushort(__float2bfloat16_rn(vp))) : "memory");
                                } else {
                                    asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(pn), "f"(vn) : "memory");
                                    asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(pp), "f"(vp) : "memory");
                                }
                                asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(pn) : "r"(Mi), "n"((int)sizeof(OT)));
                                asm("mad.wide.s32 %0, %1, %2, %0;" : "+l"(pp) : "r"(-Mi), "n"((int)sizeof(OT)));
                            }
                        } else {
#pragma unroll
                            for (int pr = 0; pr < NCH; ++pr) {
#pragma unroll
                                for (int e = 0; e < 2; ++e) {
                                    const int el = 2 * pr + e;
                                    if (el < cnt_n) st_cs_at<OT>(out, (uint32_t)(rg.x + el) * Mu, pw[pass][4 * pr + e]);
                                    if (el < cnt_p) st_cs_at<OT>(out, (uint32_t)(rg.z + cnt_p - 1 - el) * Mu, pw[pass][4 * pr + 2 + e]);
                                }
                            }
                        }
                    }
                    if (mx2[pass] > thr && col0 + lt < p.M && 2 * cg * NCH < p.nzg)
                        flag_candidate(p.search.cand, p.search.cand_count, p.search.cand_capacity,
                                       grp * p.nzg + 2 * cg * NCH, (int)(col0 + lt), mx2[pass]);
                };
                if constexpr (sizeof(OT) == 2) {
                    direct_pass(0);
                    direct_pass(1);
                    continue;
                }
                if (MODE == TB_RECHECK && smem_strip) {
                    // powers -> the strip: every bin of the listed tile, the one adjacent bin of a neighbour tile
                    const int scol = tile == centre ? 1 + lt : tile < centre ? (lt == TC_TILE - 1 ? 0 : -1) : (lt == 0 ? TC_TILE + 1 : -1);
                    if (scol >= 0) {
                        float *const S = reinterpret_cast<float *>(smem + L.off_stage) + scol;
#pragma unroll
                        for (int pass = 0; pass < 2; ++pass) {
                            const int4 rg = rg2[pass];
                            const int cnt_n = rg.y & 0xFFFF, cnt_p = rg.w & 0xFFFF;
#pragma unroll
                            for (int pr = 0; pr < NCH; ++pr) {
#pragma unroll
                                for (int e = 0; e < 2; ++e) {
                                    const int el = 2 * pr + e;
                                    if (el < cnt_n) S[(rg.x + el) * TB_STRIP_W] = pw[pass][4 * pr + e];
                                    if (el < cnt_p) S[(rg.z + cnt_p - 1 - el) * TB_STRIP_W] = pw[pass][4 * pr + 2 + e];
                                }
                            }
                        }
                    }
                    continue;
                }
                // ---- registers -> staging rows -> one tensor-map box per run
#pragma unroll
                for (int pass = 0; pass < 2; ++pass) {
                    const int cg = 2 * half + pass;
                    const int4 rg = rg2[pass];
                    // staging block (cg, stage) last fed this issuer's store of two commits ago (tile t-2, same
                    // pass): at most the newest group may still be reading shared memory
                    if (issuer) bulk_wait_read<1>();
                    named_bar_sync(bar_id, 128);
                    unsigned char *const stage_buf = smem + L.off_stage + (size_t)(SETS * cg + sblk) * L.stage_cg_bytes;
                    OT *const sb = reinterpret_cast<OT *>(stage_buf) + lt;
#pragma unroll
                    for (int pr = 0; pr < NCH; ++pr) {
                        sb[(2 * pr) * TC_TILE] = (OT)pw[pass][4 * pr];           // float -> bf16: round to nearest even
                        sb[(2 * pr + 1) * TC_TILE] = (OT)pw[pass][4 * pr + 1];
                        sb[(NC - 1 - 2 * pr) * TC_TILE] = (OT)pw[pass][4 * pr + 2];
                        sb[(NC - 2 - 2 * pr) * TC_TILE] = (OT)pw[pass][4 * pr + 3];
                    }
                    fence_proxy_async();                    // staging writes -> visible to the bulk copy engine
                    named_bar_sync(bar_id, 128);
                    if (issuer) {
                        const uint32_t sst = smem_u32(stage_buf);
                        // TB_PLANE: the planes as [batch K rows][M bins]; TB_RECHECK: this CTA's strip of scratch,
                        // [gridDim.x K rows][FDAS_TC_STRIP bins], tile j of the item in bins 128 j ..
                        const int row_s = MODE == TB_RECHECK ? (int)blockIdx.x * p.K : (int)ser * p.K;
                        const int col_s = MODE == TB_RECHECK ? tile * TC_TILE : (int)col0;
                        // one box per run: warp q = 0 pushes the -|z| rows, warp q = 1 the +|z| rows
                        const int cnt = (q ? rg.w : rg.y) & 0xFFFF, box = (q ? rg.w : rg.y) >> 16;
                        if (cnt > 0)
                            tensor_store(&maps.m[box], sst + (q ? (uint32_t)(NC - cnt) * ROWB : 0u), col_s,
                                         row_s + (q ? rg.z : rg.x));
                        bulk_commit();                      // one group per pass, empty or not: bulk_wait_read<1> counts them
                    }
                    if (MODE == TB_PLANE && mx2[pass] > thr && col0 + lt < p.M && 2 * cg * NCH < p.nzg)
                        flag_candidate(p.search.cand, p.search.cand_count, p.search.cand_capacity,
                                       grp * p.nzg + 2 * cg * NCH, (int)(col0 + lt), mx2[pass]);
                }
            }
            if constexpr (MODE == TB_RECHECK) {
                // ---- the item's powers are on their way to scratch: wait for this thread's boxes, meet every other
                // thread that wrote (all template groups), apply the peak rule of fdas_peaks (reading A14) to
                // the cells of the flagged tile, meet again before the strip is overwritten
                if (smem_strip) {
                    tb_item_sync(0, TB_EPI_WARPS * 32);
                    const float *S = reinterpret_cast<const float *>(smem + L.off_stage);
                    const int c = threadIdx.x & (TC_TILE - 1);
                    const long long r = blk0 + (long long)centre * TC_TILE + c;
                    const bool left_ok = centre == 1, right_ok = n_tiles > centre + 1;
                    for (int k = threadIdx.x >> 7; k < p.K && r < p.M; k += TB_EPI_WARPS / 4) {
                        const float v = S[k * TB_STRIP_W + 1 + c];
                        if (!(v > thr)) continue;
                        bool ok = true;
#pragma unroll
                        for (int dk = -1; dk <= 1; ++dk) {
#pragma unroll
                            for (int dr = -1; dr <= 1; ++dr) {
                                if (dk == 0 && dr == 0) continue;
                                const int kk = k + dk, cc = c + dr;
                                if (kk < 0 || kk >= p.K || r + dr < 0 || r + dr >= p.M) continue;
                                if ((cc < 0 && !left_ok) || (cc >= TC_TILE && !right_ok)) continue;
                                const float nb = S[kk * TB_STRIP_W + 1 + cc];
                                const bool precedes = (dk < 0) || (dk == 0 && dr < 0);
                                ok = ok && (precedes ? (v > nb) : (v >= nb));
                            }
                        }
                        if (ok) {
                            const int slot = atomicAdd(p.search.counts + ser, 1);
                            if (slot < p.search.capacity) {
                                fdas_peak_t rec;
                                rec.z_index = k;
                                rec.r = (int32_t)r;
                                rec.power = v;
                                p.search.peaks[(size_t)ser * p.search.capacity + slot] = rec;
                            }
                        }
                    }
                    if (threadIdx.x == 0) p.search.tile_flags[__ldcg(p.search.tile_list + it)] = 0;
                    tb_item_sync(0, TB_EPI_WARPS * 32);
                    continue;
                }
                if (issuer) bulk_wait_all();
                __threadfence();
                tb_item_sync(p.clustered, TB_EPI_WARPS * 32);
                {
                    const int G = (int)gridDim.y;
                    const int k_lo = (int)((long long)p.K * grp / G), k_hi = (int)((long long)p.K * (grp + 1) / G);
                    const float *S = p.search.scratch + (size_t)blockIdx.x * p.K * FDAS_TC_STRIP;
                    const long long r_first = blk0;                    // plane bin of strip column 0
                    const int c_lo = centre * TC_TILE, c_end = n_tiles * TC_TILE;
                    // thread -> one bin of the tile and every (TB_EPI_WARPS / 4)-th row; the loads of eight rows are in
                    // flight together (the strip is in L2: ~1 us per dependent load otherwise)
                    constexpr int RPP = TB_EPI_WARPS / 4, UB = 8;
                    const int c = c_lo + (threadIdx.x & (TC_TILE - 1));
                    const long long r = r_first + c;
                    for (int kb = k_lo + (threadIdx.x >> 7); kb < k_hi && r < p.M; kb += UB * RPP) {
                        float vv[UB];
#pragma unroll
                        for (int u = 0; u < UB; ++u)
                            vv[u] = kb + u * RPP < k_hi ? __ldcg(S + (size_t)(kb + u * RPP) * FDAS_TC_STRIP + c) : -__int_as_float(0x7f800000);
#pragma unroll
                        for (int u = 0; u < UB; ++u) {
                            const float v = vv[u];
                            if (!(v > thr)) continue;
                            const int k = kb + u * RPP;
                            bool ok = true;
#pragma unroll
                            for (int dk = -1; dk <= 1; ++dk) {
#pragma unroll
                                for (int dr = -1; dr <= 1; ++dr) {
                                    if (dk == 0 && dr == 0) continue;
                                    const int kk = k + dk, cc = c + dr;
                                    if (kk < 0 || kk >= p.K || cc < 0 || cc >= c_end || r + dr < 0 || r + dr >= p.M) continue;
                                    const float nb = __ldcg(S + (size_t)kk * FDAS_TC_STRIP + cc);
                                    const bool precedes = (dk < 0) || (dk == 0 && dr < 0);
                                    ok = ok && (precedes ? (v > nb) : (v >= nb));
                                }
                            }
                            if (ok) {
                                const int slot = atomicAdd(p.search.counts + ser, 1);
                                if (slot < p.search.capacity) {
                                    fdas_peak_t rec;
                                    rec.z_index = k;
                                    rec.r = (int32_t)r;
                                    rec.power = v;
                                    p.search.peaks[(size_t)ser * p.search.capacity + slot] = rec;
                                }
                            }
                        }
                    }
                    if (threadIdx.x == 0 && grp == 0) p.search.tile_flags[__ldcg(p.search.tile_list + it)] = 0;   // flags are all zero again after this launch
                }
                tb_item_sync(p.clustered, TB_EPI_WARPS * 32);
            }
        }
        if (issuer) bulk_wait_all();
    } else if (warp == TB_MMA_WARP) {
        // =========================== MMA issuer ===========================
        mma_issuer<NT, SPLIT, MODE>(p, s_base, L.off_z, L.z_buf_bytes, L.z_part_bytes, z_full, z_empty, t_full, t_empty,
                                    __shfl_sync(0xffffffffu, tmem_base, 0), n_items, cta);
    } else {
        // =========================== loader ===========================
        spectrum_loader<SPLIT, MODE>(p, smem, L.off_xs, L.xs_part_bytes, L.xn, L.off_z, L.z_buf_bytes, L.z_part_bytes, L.zr,
                                     z_full, z_empty, threadIdx.x - TB_LOAD_WARP0 * 32, n_items, cta, first_a, first_b);
    }

    tc_fence_before();
    __syncthreads();
    if (warp == TB_MMA_WARP) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc(tmem_base, TC_TMEM_COLS);
    }
}

}  // namespace
