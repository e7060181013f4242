// fdas_peaks.cu -- threshold + local-maximum pass over the power plane (include/fdas.h:
// fdas_peaks; reading A14).
//
// One streaming read of the plane (K*M elements).  Cells above the threshold are rare
// (noise is exponential), so the 8-neighbour test runs only for those and the
// pass is bound by the HBM read: 128-bit loads, grid sized to the SM count.
#include "fdas_internal.h"

namespace {

template <typename PT>
__device__ __forceinline__ void test_cell(const PT *__restrict__ P, int K, long long M, int k, long long r, PT v,
                                          float thr, fdas_peak_t *peaks, int capacity, int *count)
{
    if (!(v > (PT)thr)) return;
    bool ok = true;
#pragma unroll
    for (int dk = -1; dk <= 1; ++dk) {
#pragma unroll
        for (int dr = -1; dr <= 1; ++dr) {
            if (dk == 0 && dr == 0) continue;
            const int kk = k + dk;
            const long long rr = r + dr;
            if (kk < 0 || kk >= K || rr < 0 || rr >= M) continue;
            const PT n = P[(size_t)kk * M + rr];
            const bool precedes = (dk < 0) || (dk == 0 && dr < 0);
            ok = ok && (precedes ? (v > n) : (v >= n));
        }
    }
    if (ok) {
        const int slot = atomicAdd(count, 1);
        if (slot < capacity) {
            fdas_peak_t rec;
            rec.z_index = k;
            rec.r = (int32_t)r;
            rec.power = (float)v;
            peaks[slot] = rec;
        }
    }
}

template <typename PT, typename VT, int NE>
__global__ void __launch_bounds__(256)
fdas_peaks_kernel(const PT *__restrict__ P, int K, long long M, float thr, fdas_peak_t *peaks, int capacity,
                  int *count)
{
    const long long total = (long long)K * M;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (M % NE == 0) {
        const VT *PV = reinterpret_cast<const VT *>(P);
        const long long nv = total / NE;
        for (long long q = tid; q < nv; q += stride) {
            union { VT v; PT e[NE]; } u;
            u.v = __ldcs(PV + q);   // 128-bit streaming load
            PT m = u.e[0];
#pragma unroll
            for (int c = 1; c < NE; ++c) m = max(m, u.e[c]);
            if (m > (PT)thr) {
                const long long e0 = q * NE;
                const int k = (int)(e0 / M);
                const long long r = e0 - (long long)k * M;
#pragma unroll
                for (int c = 0; c < NE; ++c) test_cell<PT>(P, K, M, k, r + c, u.e[c], thr, peaks, capacity, count);
            }
        }
    } else {
        for (long long e = tid; e < total; e += stride) {
            const int k = (int)(e / M);
            test_cell<PT>(P, K, M, k, e - (long long)k * M, P[e], thr, peaks, capacity, count);
        }
    }
}

}  // namespace

int fdas_launch_peaks(fdas_plan *p, const void *plane, float thr, fdas_peak_t *peaks, int capacity, int *count,
                      cudaStream_t st)
{
    FDAS_CUDA_TRY(p, cudaMemsetAsync(count, 0, sizeof(int), st));
    const long long total = (long long)p->K * p->M;
    long long want = (total / 4 + 255) / 256;
    const long long cap = (long long)p->num_sms * 8;   // 8 resident CTAs of 256 threads per SM
    const int grid = (int)(want < cap ? (want > 0 ? want : 1) : cap);
    if (p->precision == FDAS_F64)
        fdas_peaks_kernel<double, double2, 2><<<grid, 256, 0, st>>>((const double *)plane, p->K, p->M, thr, peaks, capacity, count);
    else
        fdas_peaks_kernel<float, float4, 4><<<grid, 256, 0, st>>>((const float *)plane, p->K, p->M, thr, peaks, capacity, count);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
