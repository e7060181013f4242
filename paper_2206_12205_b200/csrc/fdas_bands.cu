// fdas_bands.cu -- harmonic-band maxima of the plane (include/fdas.h: fdas_band_max).
//
// PAPER.md:186-199, section 4.3 and Table 3: the plane is split into bands derived from the
// fundamental frequency f -- fundamental [0, 1.5 f], N-th harmonic ((N + 0.5) f, (N + 1.5) f] --
// and "the n-th harmonic is taken to be the highest point in the n-th band".  Ties (the paper is
// silent; reading A24): the first cell in (k, r) order.
//
// Two small kernels: (1) every block scans a slice of one band's columns over all K rows with
// coalesced row-wise reads and leaves its best (value, linear index); (2) one block per band
// reduces those.  Read-bound: each plane element inside a band is read once.
#include <math.h>
#include "fdas_internal.h"

namespace {

struct bm_bf16 {
    unsigned short bits;
};
template <typename T> struct bm_elem {
    static __device__ __forceinline__ double load(const T *p) { return (double)__ldg(p); }
};
template <> struct bm_elem<bm_bf16> {
    static __device__ __forceinline__ double load(const bm_bf16 *p)
    {
        return (double)__uint_as_float((unsigned)__ldg(reinterpret_cast<const unsigned short *>(p)) << 16);
    }
};

template <typename T> struct bm_cmp { using type = float; };
template <> struct bm_cmp<double> { using type = double; };

struct Best {
    double v;
    long long idx;   // k * M + r; -1 = none
};
__device__ __forceinline__ Best better(Best a, Best b)
{
    if (b.idx < 0) return a;
    if (a.idx < 0) return b;
    if (b.v > a.v || (b.v == a.v && b.idx < a.idx)) return b;
    return a;
}
__device__ __forceinline__ Best block_best(Best mine, Best *sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        Best other;
        other.v = __shfl_xor_sync(0xffffffffu, mine.v, o);
        other.idx = __shfl_xor_sync(0xffffffffu, mine.idx, o);
        mine = better(mine, other);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) sh[warp] = mine;
    __syncthreads();
    if (warp == 0) {
        mine = lane < (int)(blockDim.x >> 5) ? sh[lane] : Best{0.0, -1};
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            Best other;
            other.v = __shfl_xor_sync(0xffffffffu, mine.v, o);
            other.idx = __shfl_xor_sync(0xffffffffu, mine.idx, o);
            mine = better(mine, other);
        }
    }
    return mine;   // valid in thread 0
}

constexpr int BM_SLICE = 512;   // columns per block of fdas_band_scan_kernel (two per thread)
// band n covers bins lo[n]..hi[n] (host-computed, clipped; lo > hi = empty)
struct BandBounds {
    long long lo[FDAS_MAX_BANDS], hi[FDAS_MAX_BANDS];
};
template <typename T>
__global__ void __launch_bounds__(256) fdas_band_scan_kernel(const T *__restrict__ P, int K, long long M, const BandBounds bb,
                                                             Best *__restrict__ partial)
{
    __shared__ Best sh[8];
    const int band = blockIdx.y;
    const long long r0 = bb.lo[band], r1 = bb.hi[band];
    Best mine{0.0, -1};
    if (r0 <= r1) {
        // this block's slice of the band's columns: BM_SLICE columns starting at a multiple of BM_SLICE (so that every
        // row segment starts on a 128-byte line), clipped to the band; every row of the slice is read contiguously
        const long long a0 = (r0 / BM_SLICE + blockIdx.x) * BM_SLICE;
        const long long c0 = a0 < r0 ? r0 : a0, c1 = min(a0 + BM_SLICE, r1 + 1);
        // the first cell (in (k, r) order) of the largest value; compared in the plane's own type (float for float and bf16
        // planes: fp64 compares run at a fraction of the rate)
        using CT = typename bm_cmp<T>::type;
        CT bv = 0;
        long long bi = -1;
        auto take = [&](CT v, long long idx) {
            if (bi < 0 || v > bv || (v == bv && idx < bi)) {
                bv = v;
                bi = idx;
            }
        };
        // a thread owns columns a0 + tid and a0 + tid + 256 and walks down them with the loads of ROWS rows of both in
        // flight: the walk is bound by the latency of its loads, not by instruction issue.  Measured on the 97 x 2^22 plane,
        // 16 bands of 1e5 bins: float 0.138 ms with four rows, 0.157 with eight; bf16 0.128 / 0.114 ms.
        constexpr int ROWS = sizeof(T) == 2 ? 8 : 4;
        const long long ra = a0 + threadIdx.x, rb = ra + 256;
        const bool has_a = ra >= c0 && ra < c1, has_b = rb >= c0 && rb < c1;
        if (has_a && has_b) {
            int k = 0;
            for (; k + ROWS <= K; k += ROWS) {
                CT va[ROWS], vb[ROWS];
#pragma unroll
                for (int j = 0; j < ROWS; ++j) {
                    va[j] = (CT)bm_elem<T>::load(P + (size_t)(k + j) * M + ra);
                    vb[j] = (CT)bm_elem<T>::load(P + (size_t)(k + j) * M + rb);
                }
#pragma unroll
                for (int j = 0; j < ROWS; ++j) {
                    take(va[j], (long long)(k + j) * M + ra);
                    take(vb[j], (long long)(k + j) * M + rb);
                }
            }
            for (; k < K; ++k) {
                take((CT)bm_elem<T>::load(P + (size_t)k * M + ra), (long long)k * M + ra);
                take((CT)bm_elem<T>::load(P + (size_t)k * M + rb), (long long)k * M + rb);
            }
        } else if (has_a || has_b) {
            const long long r = has_a ? ra : rb;
            int k = 0;
            for (; k + ROWS <= K; k += ROWS) {
                CT v[ROWS];
#pragma unroll
                for (int j = 0; j < ROWS; ++j) v[j] = (CT)bm_elem<T>::load(P + (size_t)(k + j) * M + r);
#pragma unroll
                for (int j = 0; j < ROWS; ++j) take(v[j], (long long)(k + j) * M + r);
            }
            for (; k < K; ++k) take((CT)bm_elem<T>::load(P + (size_t)k * M + r), (long long)k * M + r);
        }
        mine = Best{(double)bv, bi};
    }
    mine = block_best(mine, sh);
    if (threadIdx.x == 0) partial[(size_t)band * gridDim.x + blockIdx.x] = mine;
}

__global__ void __launch_bounds__(256) fdas_band_reduce_kernel(const Best *__restrict__ partial, int n_partial, long long M,
                                                               fdas_peak_t *__restrict__ out)
{
    __shared__ Best sh[8];
    Best mine{0.0, -1};
    for (int i = threadIdx.x; i < n_partial; i += blockDim.x) mine = better(mine, partial[(size_t)blockIdx.x * n_partial + i]);
    mine = block_best(mine, sh);
    if (threadIdx.x == 0) {
        fdas_peak_t rec;
        rec.z_index = mine.idx < 0 ? -1 : (int32_t)(mine.idx / M);
        rec.r = mine.idx < 0 ? -1 : (int32_t)(mine.idx % M);
        rec.power = mine.idx < 0 ? 0.f : (float)mine.v;
        out[blockIdx.x] = rec;
    }
}

}  // namespace

int fdas_launch_band_max(fdas_plan *p, const void *plane, double f_bin, int n_bands, fdas_peak_t *out, cudaStream_t st)
{
    BandBounds bb;
    for (int n = 0; n < n_bands; ++n) {
        // Table 3: fundamental [0, 1.5 f]; band n ((n + 0.5) f, (n + 1.5) f], upper bound inclusive
        bb.lo[n] = n == 0 ? 0 : (long long)floor((n + 0.5) * f_bin) + 1;
        const long long hi = (long long)floor((n + 1.5) * f_bin);
        bb.hi[n] = hi > p->M - 1 ? p->M - 1 : hi;
    }
    // blocks per band: the slices of BM_SLICE columns the widest band touches (blocks beyond a band's last slice report nothing)
    long long nblk_ll = 1;
    for (int n = 0; n < n_bands; ++n)
        if (bb.lo[n] <= bb.hi[n]) {
            const long long need_n = bb.hi[n] / BM_SLICE - bb.lo[n] / BM_SLICE + 1;
            if (need_n > nblk_ll) nblk_ll = need_n;
        }
    const int nblk = (int)nblk_ll;
    const size_t need = (size_t)n_bands * nblk * sizeof(Best);
    if (need > p->band_scratch_bytes) {
        cudaFree(p->band_scratch);
        p->band_scratch = NULL;
        p->band_scratch_bytes = 0;
        FDAS_CUDA_TRY(p, cudaMalloc(&p->band_scratch, need));
        p->band_scratch_bytes = need;
    }
    Best *partial = static_cast<Best *>(p->band_scratch);
    const dim3 grid((unsigned)nblk, (unsigned)n_bands);
    if (p->precision == FDAS_F64)
        fdas_band_scan_kernel<double><<<grid, 256, 0, st>>>((const double *)plane, p->K, p->M, bb, partial);
    else if (p->plane_bf16)
        fdas_band_scan_kernel<bm_bf16><<<grid, 256, 0, st>>>((const bm_bf16 *)plane, p->K, p->M, bb, partial);
    else
        fdas_band_scan_kernel<float><<<grid, 256, 0, st>>>((const float *)plane, p->K, p->M, bb, partial);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    fdas_band_reduce_kernel<<<n_bands, 256, 0, st>>>(partial, nblk, p->M, out);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 2;
    return FDAS_OK;
}
