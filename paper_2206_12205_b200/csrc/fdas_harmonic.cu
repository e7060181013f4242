// fdas_harmonic.cu -- harmonic sum over the f-fdot plane (include/fdas.h: fdas_harmonic_sum).
//
// a pulsar "will appear as a peak on this plane, with diminishing harmonics at integer
// multiples of both f and fdot.  The summed height (power) of the peak and harmonics is typically
// used to calculate the signal-to-noise ratio"; "a harmonic sum algorithm is used to
// gather the power from all harmonics into a single detection".  Reading A23: the
// plain definition
//      S_H[k][r] = sum_{h=1..H} P[k0 + h (k - k0)][h r],     k0 = row of z = 0,
// skipping terms whose row or bin falls outside the plane.
//
// A gather bound by HBM reads: harmonic h touches every 32-byte sector of row k0 + h (k - k0) up
// to bin M-1 (stride-h elements, h <= 8 elements per sector), so one launch reads about
// sum_h (fraction of rows in range) planes and writes one.  Each thread owns 4 consecutive bins of
// one row: one 128-bit load for h = 1, 4 scalar read-only loads per further harmonic (a warp's
// loads of one harmonic cover a contiguous span of 128 h elements), one 128-bit streaming store.
#include "fdas_internal.h"

namespace {

struct bf16bits {
    unsigned short bits;
};
// read-only load of one plane element, widened to the arithmetic type
template <typename T> struct hs_elem {
    static __device__ __forceinline__ T load(const T *p) { return __ldg(p); }
};
template <> struct hs_elem<bf16bits> {
    static __device__ __forceinline__ float load(const bf16bits *p)
    {
        return __uint_as_float((unsigned)__ldg(reinterpret_cast<const unsigned short *>(p)) << 16);
    }
};

// DRIFT (fdas_harmonic_sum_drift, reading A26): harmonic h contributes the largest
// power of its quantisation window |dk|, |dr| <= h/2 around (k0 + h (k - k0), h r) instead of that cell alone.
template <typename IT, typename OT, bool DRIFT>
__global__ void __launch_bounds__(256) fdas_harmonic_sum_kernel(const IT *__restrict__ P, OT *__restrict__ S, int K, long long M,
                                                                int k0, int H)
{
    const int k = blockIdx.y;
    const long long quads = (M + 3) / 4;
    const IT *row1 = P + (size_t)k * M;
    OT *out = S + (size_t)k * M;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < quads; q += (long long)gridDim.x * blockDim.x) {
        const long long r = 4 * q;
        OT acc[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[j] = r + j < M ? (OT)hs_elem<IT>::load(row1 + r + j) : (OT)0;
        for (int h = 2; h <= H; ++h) {
            const long long kh = (long long)k0 + (long long)h * (k - k0);
            if (kh < 0 || kh >= K) continue;
            if (r * h >= M) break;                     // this and every further harmonic start beyond the plane
            const IT *rowh = P + (size_t)kh * M;
            if (!DRIFT) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const long long x = (r + j) * h;
                    if (x < M) acc[j] += (OT)hs_elem<IT>::load(rowh + x);
                }
            } else {
                const int t = h >> 1;
                const int dk0 = kh - t < 0 ? (int)-kh : -t, dk1 = kh + t >= K ? (int)(K - 1 - kh) : t;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const long long x = (r + j) * h;
                    if (x >= M) continue;
                    const long long x0 = x - t < 0 ? 0 : x - t, x1 = x + t >= M ? M - 1 : x + t;
                    OT best = (OT)hs_elem<IT>::load(rowh + x);
                    for (int dk = dk0; dk <= dk1; ++dk) {
                        const IT *rw = rowh + (long long)dk * M;
                        for (long long xx = x0; xx <= x1; ++xx) best = max(best, (OT)hs_elem<IT>::load(rw + xx));
                    }
                    acc[j] += best;
                }
            }
        }
        if (r + 3 < M && (M & 3) == 0 && sizeof(OT) == 4) {
            __stcs(reinterpret_cast<float4 *>(out + r), make_float4((float)acc[0], (float)acc[1], (float)acc[2], (float)acc[3]));
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (r + j < M) out[r + j] = acc[j];
        }
    }
}

// Drift-tolerant form, tiled: CTA = (row k, 1024 output bins).  For every harmonic the plane elements its windows cover
// form ONE contiguous span of rows kh - t .. kh + t (windows of 2t + 1 >= h bins at stride h tile the row), so the
// window maximum is separable: a coalesced pass takes the maximum over the rows of the span into shared memory, then
// every output takes the maximum of its 2t + 1 consecutive entries.  (2t + 1) h coalesced loads per output instead of
// (2t + 1)^2 scattered ones; maxima are exact, so the result is bit-identical to the gather form.  blockIdx.x = k
// (fastest) keeps the rows that share plane rows -- output rows k and k + 1 overlap in 2t + 1 - h of them -- together
// in L2.
constexpr int HD_THREADS = 256, HD_OUT = 4, HD_TILE = HD_THREADS * HD_OUT, HD_SPAN = 4096 + 64;

template <typename IT, typename OT>
__global__ void __launch_bounds__(HD_THREADS) fdas_harmonic_drift_kernel(const IT *__restrict__ P, OT *__restrict__ S, int K, long long M,
                                                                         int k0, int H)
{
    __shared__ __align__(16) OT buf[HD_SPAN];
    const int k = blockIdx.x;
    const long long r0 = (long long)blockIdx.y * HD_TILE;
    const IT *row1 = P + (size_t)k * M;
    OT acc[HD_OUT];
#pragma unroll
    for (int j = 0; j < HD_OUT; ++j) {
        const long long r = r0 + threadIdx.x + HD_THREADS * j;      // thread -> bins r0 + tid + 256 j: coalesced, stride-h smem reads
        acc[j] = r < M ? (OT)hs_elem<IT>::load(row1 + r) : (OT)0;
    }
    for (int h = 2; h <= H; ++h) {
        const long long kh = (long long)k0 + (long long)h * (k - k0);
        if (kh < 0 || kh >= K) continue;
        if (r0 * h >= M) break;                        // this and every further harmonic start beyond the plane
        const int t = h >> 1;
        const int dk0 = kh - t < 0 ? (int)-kh : -t, dk1 = kh + t >= K ? (int)(K - 1 - kh) : t;
        const IT *rowh = P + (size_t)kh * M;
        const int chunk = (HD_SPAN - 2 * t - 16) / h < HD_TILE ? (HD_SPAN - 2 * t - 16) / h : HD_TILE;   // outputs per span (7 bins of alignment slack at either end)
        for (int c0 = 0; c0 < HD_TILE; c0 += chunk) {
            const long long rc = r0 + c0;                              // first output bin of this chunk
            if (rc * h >= M) break;
            const int nout = HD_TILE - c0 < chunk ? HD_TILE - c0 : chunk;
            const long long x_lo = rc * h - t < 0 ? 0 : rc * h - t;
            long long x_base;                                          // plane bin of buf[0]
            long long x_hi = (rc + nout - 1) * h + t;
            if (x_hi > M - 1) x_hi = M - 1;
            const int span = (int)(x_hi - x_lo + 1);
            if (sizeof(IT) == 4 && sizeof(OT) == 4 && (M & 3) == 0) {
                // float planes with 16-byte aligned rows: 128-bit loads from the aligned start of the span (buf index 0 = x_al)
                const long long x_al = x_lo & ~3LL;
                const int nq = (int)((x_hi - x_al) / 4 + 1);
                for (int i = threadIdx.x; i < nq; i += HD_THREADS) {
                    const float4 *src = reinterpret_cast<const float4 *>(rowh + (long long)dk0 * M + x_al) + i;
                    float4 v = __ldg(src);
                    for (int dk = dk0 + 1; dk <= dk1; ++dk) {
                        const float4 w = __ldg(reinterpret_cast<const float4 *>(rowh + (long long)dk * M + x_al) + i);
                        v.x = fmaxf(v.x, w.x); v.y = fmaxf(v.y, w.y); v.z = fmaxf(v.z, w.z); v.w = fmaxf(v.w, w.w);
                    }
                    reinterpret_cast<float4 *>(buf)[i] = v;
                }
                x_base = x_al;
            } else if (sizeof(IT) == 2 && (M & 7) == 0) {
                // bf16-stored planes with 16-byte aligned rows: eight elements per load, widened (bits << 16) and compared
                // as floats (2.78 ms with one 16-bit load per element, the float plane's 1.75 ms being the faster one)
                if constexpr (sizeof(IT) == 2) {
                    const long long x_al = x_lo & ~7LL;
                    const int nq = (int)((x_hi - x_al) / 8 + 1);
                    const size_t M8 = (size_t)(M >> 3);
                    for (int i = threadIdx.x; i < nq; i += HD_THREADS) {
                        const uint4 *src = reinterpret_cast<const uint4 *>(rowh + (long long)dk0 * M + x_al) + i;
                        float f[8];
                        {
                            const uint4 v = __ldg(src);
                            const unsigned w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                f[2 * e] = __uint_as_float(w4[e] << 16);
                                f[2 * e + 1] = __uint_as_float(w4[e] & 0xFFFF0000u);
                            }
                        }
                        for (int dk = dk0 + 1; dk <= dk1; ++dk) {
                            const uint4 v = __ldg(src + (size_t)(dk - dk0) * M8);
                            const unsigned w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                f[2 * e] = fmaxf(f[2 * e], __uint_as_float(w4[e] << 16));
                                f[2 * e + 1] = fmaxf(f[2 * e + 1], __uint_as_float(w4[e] & 0xFFFF0000u));
                            }
                        }
                        reinterpret_cast<float4 *>(buf)[2 * i] = make_float4(f[0], f[1], f[2], f[3]);
                        reinterpret_cast<float4 *>(buf)[2 * i + 1] = make_float4(f[4], f[5], f[6], f[7]);
                    }
                    x_base = x_al;
                }
            } else {
                for (int i = threadIdx.x; i < span; i += HD_THREADS) {
                    OT v = (OT)hs_elem<IT>::load(rowh + (long long)dk0 * M + x_lo + i);
                    for (int dk = dk0 + 1; dk <= dk1; ++dk) v = max(v, (OT)hs_elem<IT>::load(rowh + (long long)dk * M + x_lo + i));
                    buf[i] = v;
                }
                x_base = x_lo;
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < HD_OUT; ++j) {
                const int o = threadIdx.x + HD_THREADS * j - c0;       // output index inside the chunk
                if (o < 0 || o >= nout) continue;
                const long long x = (rc + o) * h;
                if (x >= M) continue;
                const long long a = x - t < 0 ? 0 : x - t, b = x + t > M - 1 ? M - 1 : x + t;
                OT best = buf[a - x_base];
                for (long long xx = a + 1; xx <= b; ++xx) best = max(best, buf[xx - x_base]);
                acc[j] += best;
            }
            __syncthreads();
        }
    }
#pragma unroll
    for (int j = 0; j < HD_OUT; ++j) {
        const long long r = r0 + threadIdx.x + HD_THREADS * j;
        if (r < M) S[(size_t)k * M + r] = acc[j];
    }
}

}  // namespace

template <bool DRIFT>
static void launch_hs(fdas_plan *p, const void *plane, void *sum, int n_harmonics, int k0, dim3 grid, cudaStream_t st)
{
    if (p->precision == FDAS_F64)
        fdas_harmonic_sum_kernel<double, double, DRIFT><<<grid, 256, 0, st>>>((const double *)plane, (double *)sum, p->K, p->M, k0, n_harmonics);
    else if (p->plane_bf16)
        fdas_harmonic_sum_kernel<bf16bits, float, DRIFT><<<grid, 256, 0, st>>>((const bf16bits *)plane, (float *)sum, p->K, p->M, k0, n_harmonics);
    else
        fdas_harmonic_sum_kernel<float, float, DRIFT><<<grid, 256, 0, st>>>((const float *)plane, (float *)sum, p->K, p->M, k0, n_harmonics);
}

int fdas_launch_harmonic_sum(fdas_plan *p, const void *plane, void *sum, int n_harmonics, int k0, int drift, cudaStream_t st)
{
    const long long quads = (p->M + 3) / 4;
    long long bx = (quads + 255) / 256;
    const long long cap = (long long)p->num_sms * 8;
    if (bx * p->K > cap) bx = (cap + p->K - 1) / p->K;
    if (bx < 1) bx = 1;
    const dim3 grid((unsigned)bx, (unsigned)p->K);
    const long long tiles = (p->M + HD_TILE - 1) / HD_TILE;
    if (drift && tiles <= 65535) {
        const dim3 gd((unsigned)p->K, (unsigned)tiles);
        if (p->precision == FDAS_F64)
            fdas_harmonic_drift_kernel<double, double><<<gd, HD_THREADS, 0, st>>>((const double *)plane, (double *)sum, p->K, p->M, k0, n_harmonics);
        else if (p->plane_bf16)
            fdas_harmonic_drift_kernel<bf16bits, float><<<gd, HD_THREADS, 0, st>>>((const bf16bits *)plane, (float *)sum, p->K, p->M, k0, n_harmonics);
        else
            fdas_harmonic_drift_kernel<float, float><<<gd, HD_THREADS, 0, st>>>((const float *)plane, (float *)sum, p->K, p->M, k0, n_harmonics);
    } else if (drift) launch_hs<true>(p, plane, sum, n_harmonics, k0, grid, st);
    else launch_hs<false>(p, plane, sum, n_harmonics, k0, grid, st);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
