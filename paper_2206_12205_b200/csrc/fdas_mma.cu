// fdas_mma.cu -- tensor-core (tcgen05 / TMEM) form of the bf16 convolution
// (include/fdas.h: fdas_convolve with FDAS_BF16 and FDAS_ALGO_MMA).
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
//      B[n][kappa] = hre_|z|[M0 - kappa] (n even) or him_|z|[M0 - kappa] (n odd)
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
// One persistent CTA per SM, warp-specialised:
//   warps 0-7   epilogue: tcgen05.ld -> |.|^2 -> st.global.cs (TMEM double-buffered)
//   warp  8     one thread issues tcgen05.mma and tcgen05.commit
//   warps 9-12  loader: spectrum block -> bf16 (RNE, reading A12) -> Z rows
#include <cuda_bf16.h>
#include <math.h>
#include <stdlib.h>
#include "fdas_internal.h"

namespace {

constexpr int TC_TILE = 128;            // outputs per MMA tile = UMMA M = TMEM lanes
constexpr int TC_EPI_WARPS = 8;
constexpr int TC_MMA_WARP = 8;
constexpr int TC_LOAD_WARP0 = 9;
constexpr int TC_LOAD_WARPS = 4;
constexpr int TC_LOAD_THREADS = 32 * TC_LOAD_WARPS;
constexpr int TC_THREADS = 32 * (TC_EPI_WARPS + 1 + TC_LOAD_WARPS);   // 416
constexpr int TC_TMEM_COLS = 512;       // whole TMEM: 2 stages x (re | im) x NT <= 128 columns
constexpr int TC_STAGE_COLS = 256;
constexpr long long TC_SPIN_LIMIT = 1LL << 26;   // a stuck pipeline traps instead of hanging the GPU

struct TcParams {
    const float2 *spectra;   // [batch][M] complex64
    float *planes;           // [batch][K][M]
    const uint4 *bmat;       // [groups][2 KS][NT] rows of 8 bf16 (the shared-memory image)
    const int2 *ktab;        // [groups][nzg]: plane rows of (+|z|, -|z|), -1 where absent
    long long M;
    int K, batch;
    int R;                   // outputs per work item (multiple of 128)
    int n_blocks;            // ceil(M / R)
    int M0;                  // m_max: T[r][kappa] = X[r - M0 + kappa]
    int KS;                  // K steps of 16 taps
    int NT;                  // UMMA N: columns per part (multiple of 16, <= 128) = 16 NCH
    int nzg;                 // |z| values per group
    int full_chunks;         // 16-column chunks whose 8 |z| entries all have both plane rows
    fdas_search_args search; // fused threshold pass (fdas_search); enabled = 0 for plain fdas_convolve
};

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
    long long spins = 0;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.b32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
        if (!done) {
            if (++spins > TC_SPIN_LIMIT) __trap();
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

// D[tmem] (+)= A[smem desc] * B[smem desc]^T, bf16 x bf16 -> fp32, M = 128, K = 16
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrives on the mbarrier once every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
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
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46);
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

// streaming store of v at base + off (plane elements): one IMAD.WIDE for the address
__device__ __forceinline__ void st_cs_at(const float *base, uint32_t off, float v)
{
    unsigned long long addr;
    asm("mad.wide.u32 %0, %1, 4, %2;" : "=l"(addr) : "r"(off), "l"(base));
    asm volatile("st.global.cs.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

constexpr uint32_t TC_NO_ROW = 0xFFFFFFFFu;   // row-offset table: this |z| has no such plane row

// |.|^2 of Y_{+|z|} and Y_{-|z|} for the eight |z| of one 16-column chunk (file header) and the
// stores.  v[0..15] = (Ure, Vre) pairs, v[16..31] = (Uim, Vim) pairs of this thread's output bin;
// o4[0..3] = row offsets (+|z|, -|z|) of two |z| each, in plane elements.
// FAST: the tile lies inside the plane and every entry has both rows -> straight-line code.
// Returns the largest power this thread stored (0 if none): the fused search flags the chunk
// when it exceeds the threshold (fdas_search).
template <bool FAST>
__device__ __forceinline__ float epilogue_chunk(const uint32_t *v, const uint4 *o4, float *out, bool ok)
{
    float mx = 0.f;
#pragma unroll
    for (int e2 = 0; e2 < 4; ++e2) {
        const uint4 o = o4[e2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int e = 2 * e2 + s;
            const uint32_t offp = s ? o.z : o.x, offm = s ? o.w : o.y;
            const float ure = __uint_as_float(v[2 * e]), vre = __uint_as_float(v[2 * e + 1]);
            const float uim = __uint_as_float(v[16 + 2 * e]), vim = __uint_as_float(v[16 + 2 * e + 1]);
            if (FAST) {
                const float a = ure - vim, b = uim + vre, c = ure + vim, d = uim - vre;
                const float pp = a * a + b * b, pm = c * c + d * d;
                st_cs_at(out, offp, pp);
                st_cs_at(out, offm, pm);
                mx = fmaxf(mx, fmaxf(pp, pm));
            } else {
                if (offp != TC_NO_ROW && ok) {
                    const float a = ure - vim, b = uim + vre;
                    const float pp = a * a + b * b;
                    st_cs_at(out, offp, pp);
                    mx = fmaxf(mx, pp);
                }
                if (offm != TC_NO_ROW && ok) {
                    const float c = ure + vim, d = uim - vre;
                    const float pm = c * c + d * d;
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
template <int NCH, int HALF>
__device__ __forceinline__ void epilogue_tile(uint32_t taddr, const uint4 *otab4, float *out, bool inside, bool ok,
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
#ifdef FDAS_MMA_DEBUG_NOSTORE
        ok = false; inside = false;
#endif
        float mx;
        if (inside && c < full_chunks) mx = epilogue_chunk<true>(v[i & 1], otab4 + 4 * c, out, true);
        else mx = epilogue_chunk<false>(v[i & 1], otab4 + 4 * c, out, ok);
        if (mx > thr)   // thr = +inf unless fdas_search
            flag_candidate(sa.cand, sa.cand_count, sa.cand_capacity, zi_group0 + 8 * c, (int)col, mx);
    }
    if (NMY == 0) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar);
    }
}

template <int NCH>
__global__ void __launch_bounds__(TC_THREADS, 1) fdas_mma_convolve_kernel(const TcParams p)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int NT = 16 * NCH;
    const TcSmem L(p.R, p.KS, NT);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = blockIdx.y;
    const long long n_items = (long long)p.batch * p.n_blocks;

    const uint32_t s_base = smem_u32(smem);
    const uint32_t bars = s_base + L.off_bars;
    // barrier slots: z_full[2] (loader -> mma), z_empty[2] (mma -> loader),
    //                t_full[2] (mma -> epilogue), t_empty[2] (epilogue -> mma)
    const uint32_t z_full = bars, z_empty = bars + 16, t_full = bars + 32, t_empty = bars + 48;
    uint32_t *holder = reinterpret_cast<uint32_t *>(smem + L.off_holder);
    uint2 *otab = reinterpret_cast<uint2 *>(smem + L.off_ktab);   // [NT/2] row offsets (+|z|, -|z|)

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
    if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0 && p.search.enabled) {
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
        for (long long it = blockIdx.x; it < n_items; it += gridDim.x) {
            const long long ser = it / p.n_blocks;
            const long long blk0 = (it % p.n_blocks) * p.R;
            const long long left = p.M - blk0;
            const int n_tiles = (int)((left < p.R ? left : p.R) + TC_TILE - 1) / TC_TILE;
            for (int tile = 0; tile < n_tiles; ++tile, ++t) {
                const uint32_t stage = t & 1, use = t >> 1;
                const long long col0 = blk0 + tile * TC_TILE;
                const long long col = col0 + q * 32 + lane;
                float *const out = p.planes + (size_t)ser * p.K * p.M + col;
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + stage * TC_STAGE_COLS;
                const bool inside = col0 + TC_TILE <= p.M;
                mbar_wait(t_full + 8 * stage, use & 1);
                tc_fence_after();
                if (half == 0)
                    epilogue_tile<NCH, 0>(taddr, otab4, out, inside, col < p.M, p.full_chunks, t_empty + 8 * stage, lane,
                                          p.search, thr, zi_group0, col);
                else
                    epilogue_tile<NCH, 1>(taddr, otab4, out, inside, col < p.M, p.full_chunks, t_empty + 8 * stage, lane,
                                          p.search, thr, zi_group0, col);
            }
        }
    } else if (warp == TC_MMA_WARP) {
        // =========================== MMA issuer ===========================
        if (lane == 0) {
            // instruction descriptor (cute::UMMA::InstrDescriptor): fp32 accumulate, bf16 A and B,
            // both K-major, N = NT, M = 128
            const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NT >> 3) << 17) |
                                   ((uint32_t)(TC_TILE >> 4) << 24);
            const uint32_t b_addr = s_base;
            const uint32_t b_lbo = (uint32_t)NT * 16u;   // next 8-tap chunk of the tap matrix
            uint32_t n = 0, t = 0;
            for (long long it = blockIdx.x; it < n_items; it += gridDim.x, ++n) {
                const uint32_t buf = n & 1, zuse = n >> 1;
                const long long blk0 = (it % p.n_blocks) * p.R;
                const long long left = p.M - blk0;
                const int n_tiles = (int)((left < p.R ? left : p.R) + TC_TILE - 1) / TC_TILE;
                mbar_wait(z_full + 8 * buf, zuse & 1);
                tc_fence_after();
                const uint32_t z_addr = s_base + L.off_z + buf * L.z_buf_bytes;
                for (int tile = 0; tile < n_tiles; ++tile, ++t) {
                    const uint32_t stage = t & 1, use = t >> 1;
                    mbar_wait(t_empty + 8 * stage, (use & 1) ^ 1);
                    tc_fence_after();
                    for (int part = 0; part < 2; ++part) {
                        const uint32_t d = tmem_base + stage * TC_STAGE_COLS + part * NT;
                        const uint32_t a0 = z_addr + part * L.z_part_bytes + (uint32_t)(tile * TC_TILE) * 16u;
                        for (int ks = 0; ks < p.KS; ++ks) {
                            const uint64_t ad = smem_desc(a0 + ks * 256u, 128u, 128u);
                            const uint64_t bd = smem_desc(b_addr + ks * 2u * b_lbo, b_lbo, 128u);
#ifndef FDAS_MMA_DEBUG_NOMMA
                            umma_bf16(d, ad, bd, idesc, ks > 0);
#else
                            (void)ad; (void)bd; (void)d;
#endif
                        }
                    }
                    umma_commit(t_full + 8 * stage);
                }
                umma_commit(z_empty + 8 * buf);
            }
        }
    } else {
        // =========================== loader ===========================
        const int lt = threadIdx.x - TC_LOAD_WARP0 * 32;
        uint32_t *xs_re = reinterpret_cast<uint32_t *>(smem + L.off_xs);
        uint32_t *xs_im = reinterpret_cast<uint32_t *>(smem + L.off_xs + L.xs_part_bytes);
        uint32_t n = 0;
        for (long long it = blockIdx.x; it < n_items; it += gridDim.x, ++n) {
            const uint32_t buf = n & 1, zuse = n >> 1;
            const long long ser = it / p.n_blocks;
            const long long g0 = (it % p.n_blocks) * p.R - p.M0;   // sample index of xs[0]
            const float2 *__restrict__ X = p.spectra + (size_t)ser * p.M;
            // phase A: spectrum block -> bf16 (round-to-nearest-even), re and im planes
            for (uint32_t pi = lt; pi < L.xn / 2; pi += TC_LOAD_THREADS) {
                const long long g = g0 + 2 * (long long)pi;
                float2 a = make_float2(0.f, 0.f), b = make_float2(0.f, 0.f);
                if (g >= 0 && g < p.M) a = __ldg(X + g);
                if (g + 1 >= 0 && g + 1 < p.M) b = __ldg(X + g + 1);
                xs_re[pi] = pack_bf16(a.x, b.x);
                xs_im[pi] = pack_bf16(a.y, b.y);
            }
            named_bar_sync(1, TC_LOAD_THREADS);
            mbar_wait<64>(z_empty + 8 * buf, (zuse & 1) ^ 1);
            // phase B: Z row i = samples i .. i+7 (16 bytes), for both parts
            unsigned char *zb = smem + L.off_z + buf * L.z_buf_bytes;
            for (uint32_t row = lt; row < L.zr; row += TC_LOAD_THREADS) {
#pragma unroll
                for (int part = 0; part < 2; ++part) {
                    const uint32_t *w = (part ? xs_im : xs_re) + (row >> 1);
                    uint4 o;
                    if (row & 1) {
                        const uint32_t w0 = w[0], w1 = w[1], w2 = w[2], w3 = w[3], w4 = w[4];
                        o.x = __byte_perm(w0, w1, 0x5432);
                        o.y = __byte_perm(w1, w2, 0x5432);
                        o.z = __byte_perm(w2, w3, 0x5432);
                        o.w = __byte_perm(w3, w4, 0x5432);
                    } else {
                        o = make_uint4(w[0], w[1], w[2], w[3]);
                    }
                    *reinterpret_cast<uint4 *>(zb + part * L.z_part_bytes + (size_t)row * 16) = o;
                }
            }
            fence_proxy_async();   // generic-proxy writes of Z -> visible to tcgen05.mma
            mbar_arrive(z_full + 8 * buf);
            named_bar_sync(1, TC_LOAD_THREADS);   // xs is rewritten by the next item
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == TC_MMA_WARP) {
        __syncwarp();
        tc_fence_after();
        tmem_dealloc(tmem_base, TC_TMEM_COLS);
    }
}

// ---- tap matrix builder -----------------------------------------------------------------
// bmat[g][q][n][e], kappa = 8 q + e, j = M0 - kappa: bf16(RNE, once from fp64) of the real
// (n even) or imaginary (n odd) part of h_{+|z|}[j] for |z| index g*nzg + n/2; zero padding.
// kref[g][zi] = (template whose fp64 taps are read, +1 if its z >= 0 else -1): h_{+|z|} = conj(h_{-|z|}).
__global__ void fdas_tapmatrix_kernel(__nv_bfloat16 *bmat, const double2 *__restrict__ taps, const int2 *__restrict__ kref,
                                      int groups, int nzg, int NT, int KS, int m_max)
{
    const size_t total = (size_t)groups * 2 * KS * NT * 8;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int e = (int)(idx % 8);
        const int n = (int)((idx / 8) % NT);
        const int qq = (int)((idx / 8 / NT) % (2 * KS));
        const int g = (int)(idx / 8 / NT / (2 * KS));
        const int j = m_max - (8 * qq + e);
        const int zi = n >> 1;
        double v = 0.0;
        if (j >= -m_max && zi < nzg) {
            const int2 kr = kref[(size_t)g * nzg + zi];
            if (kr.x >= 0) {
                const double2 h = taps[(size_t)kr.x * (2 * m_max + 1) + (m_max + j)];
                v = (n & 1) ? (double)kr.y * h.y : h.x;
            }
        }
        bmat[idx] = __double2bfloat16(v);
    }
}

}  // namespace

// Host: the |z| grouping.  Templates z_k = -zmax + k dz pair up as (k, K-1-k) when zmax is a
// multiple of dz; otherwise every template stands alone.
int fdas_mma_plan(fdas_plan *p)
{
    if (p->precision != FDAS_BF16) return FDAS_OK;
    const int K = p->K;
    const bool symmetric = fabs(-2.0 * p->zmax + (K - 1) * p->dz) <= 1e-9 * (1.0 + p->zmax);
    const int nz = symmetric ? (K + 1) / 2 : K;
    const int groups = (nz + 63) / 64;
    const int nzg = (nz + groups - 1) / groups;
    const int NT = (2 * nzg + 15) / 16 * 16;
    const int KS = (2 * p->m_max + 1 + 15) / 16;
    // row offsets k*M are 32-bit plane-element offsets inside the kernel
    p->tc_supported = (KS <= 32 && NT <= 128 && (long long)K * p->M < 0xFFFFFFFFLL);
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
            const bool neg = (-p->zmax + (double)i * p->dz) < 0.0;
            tab[i] = neg ? make_int2(-1, (int)i) : make_int2((int)i, -1);
            ref[i] = make_int2((int)i, neg ? -1 : 1);
        }
    }
    // leading 16-column chunks (8 |z| each) in which every entry has both plane rows, in every group
    p->tc_full_chunks = NT / 16;
    for (int g = 0; g < groups; ++g) {
        int lead = 0;
        while (lead < nzg && tab[(size_t)g * nzg + lead].x >= 0 && tab[(size_t)g * nzg + lead].y >= 0) ++lead;
        if (lead / 8 < p->tc_full_chunks) p->tc_full_chunks = lead / 8;
    }
    p->tc_bmat_bytes = (size_t)groups * 2 * KS * NT * 16;
    cudaError_t e;
    if ((e = cudaMalloc(&p->tc_bmat, p->tc_bmat_bytes)) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tc_ktab, n_tab * sizeof(int2))) != cudaSuccess ||
        (e = cudaMalloc((void **)&p->tc_kref, n_tab * sizeof(int2))) != cudaSuccess ||
        (e = cudaMemcpy(p->tc_ktab, tab, n_tab * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(p->tc_kref, ref, n_tab * sizeof(int2), cudaMemcpyHostToDevice)) != cudaSuccess) {
        free(tab);
        free(ref);
        p->last_err = e;
        return e == cudaErrorMemoryAllocation ? FDAS_ERR_ALLOC : FDAS_ERR_CUDA;
    }
    free(tab);
    free(ref);
    return FDAS_OK;
}

int fdas_launch_build_tapmatrix(fdas_plan *p, cudaStream_t st)
{
    if (p->precision != FDAS_BF16 || !p->tc_supported) return FDAS_OK;
    const size_t total = p->tc_bmat_bytes / 2;
    const int blocks = (int)((total + 255) / 256 < 1024 ? (total + 255) / 256 : 1024);
    fdas_tapmatrix_kernel<<<blocks, 256, 0, st>>>((__nv_bfloat16 *)p->tc_bmat, p->taps, p->tc_kref,
                                                  p->tc_groups, p->tc_nzg, p->tc_NT, p->tc_KS, p->m_max);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

template <int NCH>
static int launch_mma(fdas_plan *p, const TcParams &tp, unsigned gx, size_t smem_bytes, cudaStream_t st)
{
    auto kern = fdas_mma_convolve_kernel<NCH>;
    static size_t attr_bytes = 0;
    if (smem_bytes > attr_bytes) {
        FDAS_CUDA_TRY(p, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
        attr_bytes = smem_bytes;
    }
    kern<<<dim3(gx, p->tc_groups), TC_THREADS, smem_bytes, st>>>(tp);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

int fdas_launch_convolve_mma(fdas_plan *p, const void *spectra, void *planes, int batch, cudaStream_t st,
                             const fdas_search_args *search)
{
    if (p->precision != FDAS_BF16 || !p->tc_supported) return FDAS_ERR_UNSUPPORTED;
    // outputs per work item: the largest of 1024..128 that fits shared memory and leaves at
    // least two items per CTA
    const int sms_per_group = p->num_sms / p->tc_groups > 0 ? p->num_sms / p->tc_groups : 1;
    int R = 1024;
    for (;; R >>= 1) {
        const TcSmem L(R, p->tc_KS, p->tc_NT);
        const long long items = (long long)batch * ((p->M + R - 1) / R);
        if (R == 128 || (L.total <= 227u * 1024u && items >= 2LL * sms_per_group)) break;
    }
    const TcSmem L(R, p->tc_KS, p->tc_NT);
    if (L.total > 227u * 1024u) return FDAS_ERR_UNSUPPORTED;
    TcParams tp;
    tp.spectra = static_cast<const float2 *>(spectra);
    tp.planes = static_cast<float *>(planes);
    tp.bmat = static_cast<const uint4 *>(p->tc_bmat);
    tp.ktab = p->tc_ktab;
    tp.M = p->M;
    tp.K = p->K;
    tp.batch = batch;
    tp.R = R;
    tp.n_blocks = (int)((p->M + R - 1) / R);
    tp.M0 = p->m_max;
    tp.KS = p->tc_KS;
    tp.NT = p->tc_NT;
    tp.nzg = p->tc_nzg;
    tp.full_chunks = p->tc_full_chunks;
    if (search) tp.search = *search;
    else tp.search = fdas_search_args{0, 0.f, nullptr, nullptr, nullptr, 0, nullptr};
    const long long items = (long long)batch * tp.n_blocks;
    const unsigned gx = (unsigned)(items < sms_per_group ? items : sms_per_group);
    switch (p->tc_NT / 16) {
    case 1: return launch_mma<1>(p, tp, gx, L.total, st);
    case 2: return launch_mma<2>(p, tp, gx, L.total, st);
    case 3: return launch_mma<3>(p, tp, gx, L.total, st);
    case 4: return launch_mma<4>(p, tp, gx, L.total, st);
    case 5: return launch_mma<5>(p, tp, gx, L.total, st);
    case 6: return launch_mma<6>(p, tp, gx, L.total, st);
    case 7: return launch_mma<7>(p, tp, gx, L.total, st);
    case 8: return launch_mma<8>(p, tp, gx, L.total, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}
