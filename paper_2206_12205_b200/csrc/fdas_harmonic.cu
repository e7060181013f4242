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
    if (drift) launch_hs<true>(p, plane, sum, n_harmonics, k0, grid, st);
    else launch_hs<false>(p, plane, sum, n_harmonics, k0, grid, st);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
