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
        const long long width = r1 - r0 + 1;
        // this block's slice of the band's columns; every row of the slice is read contiguously
        const long long per = (width + gridDim.x - 1) / gridDim.x;
        const long long c0 = r0 + (long long)blockIdx.x * per, c1 = min(c0 + per, r1 + 1);
        // the first cell (in (k, r) order) of the largest value; compared in the plane's own type (float for float and bf16
        // planes: fp64 compares run at a fraction of the rate)
        using CT = typename bm_cmp<T>::type;
        CT bv = 0;
        long long bi = -1;
        // (the slice is a few hundred columns wide: a thread has one or two cells per row, so the loads of four rows are
        // put in flight together)
        for (long long r = c0 + threadIdx.x; r < c1; r += blockDim.x) {
            int k = 0;
            for (; k + 4 <= K; k += 4) {
                CT v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] = (CT)bm_elem<T>::load(P + (size_t)(k + j) * M + r);
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (bi < 0 || v[j] > bv || (v[j] == bv && (long long)(k + j) * M + r < bi)) {
                        bv = v[j];
                        bi = (long long)(k + j) * M + r;
                    }
            }
            for (; k < K; ++k) {
                const CT v = (CT)bm_elem<T>::load(P + (size_t)k * M + r);
                if (bi < 0 || v > bv || (v == bv && (long long)k * M + r < bi)) {
                    bv = v;
                    bi = (long long)k * M + r;
                }
            }
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
    const int nblk = p->num_sms * 2;                               // blocks per band
    const size_t need = (size_t)n_bands * nblk * sizeof(Best);
    if (need > p->band_scratch_bytes) {
        cudaFree(p->band_scratch);
        p->band_scratch = NULL;
        p->band_scratch_bytes = 0;
        FDAS_CUDA_TRY(p, cudaMalloc(&p->band_scratch, need));
        p->band_scratch_bytes = need;
    }
    BandBounds bb;
    for (int n = 0; n < n_bands; ++n) {
        // Table 3: fundamental [0, 1.5 f]; band n ((n + 0.5) f, (n + 1.5) f], upper bound inclusive
        bb.lo[n] = n == 0 ? 0 : (long long)floor((n + 0.5) * f_bin) + 1;
        const long long hi = (long long)floor((n + 1.5) * f_bin);
        bb.hi[n] = hi > p->M - 1 ? p->M - 1 : hi;
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
