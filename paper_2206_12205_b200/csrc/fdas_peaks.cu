// fdas_peaks.cu -- threshold + local-maximum pass over the power plane (include/fdas.h:
// fdas_peaks; reading A14).
//
// One streaming read of the plane (K*M elements).  Cells above the threshold are rare
// (noise is exponential), so the 8-neighbour test runs only for those and the
// pass is bound by the HBM read: 128-bit loads, grid sized to the SM count.
#include "fdas_internal.h"

namespace {

// Plane element types: double (FDAS_F64), float, and bf16 bit patterns (the bf16-stored plane of
// PAPER.md:91; its value is the fp32 number with those 16 bits on top -- the "quick cast").
struct bf16raw {
    unsigned short bits;
};
template <typename PT> struct elem {
    using cmp = PT;
    static __device__ __forceinline__ cmp val(PT x) { return x; }
};
template <> struct elem<bf16raw> {
    using cmp = float;
    static __device__ __forceinline__ cmp val(bf16raw x) { return __uint_as_float((unsigned)x.bits << 16); }
};

template <typename PT>
__device__ __forceinline__ void test_cell(const PT *__restrict__ P, int K, long long M, int k, long long r,
                                          typename elem<PT>::cmp v, float thr, fdas_peak_t *peaks, int capacity, int *count)
{
    using CT = typename elem<PT>::cmp;
    if (!(v > (CT)thr)) return;
    bool ok = true;
#pragma unroll
    for (int dk = -1; dk <= 1; ++dk) {
#pragma unroll
        for (int dr = -1; dr <= 1; ++dr) {
            if (dk == 0 && dr == 0) continue;
            const int kk = k + dk;
            const long long rr = r + dr;
            if (kk < 0 || kk >= K || rr < 0 || rr >= M) continue;
            const CT n = elem<PT>::val(P[(size_t)kk * M + rr]);
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
        // four 128-bit streaming loads in flight per thread; a vector holding a value above the threshold is rare
        // (a few thousand of 1e8 on config 3) and handled out of line
        constexpr int UNR = 4;
        for (long long q0 = tid; q0 < nv; q0 += UNR * stride) {
            union { VT v; PT e[NE]; } u[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j)
                if (q0 + j * stride < nv) u[j].v = __ldcs(PV + q0 + j * stride);
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const long long q = q0 + j * stride;
                if (q >= nv) break;
                using CT = typename elem<PT>::cmp;
                CT m = elem<PT>::val(u[j].e[0]);
#pragma unroll
                for (int c = 1; c < NE; ++c) m = max(m, elem<PT>::val(u[j].e[c]));
                if (m > (CT)thr) {
                    const long long e0 = q * NE;
                    const int k = (int)(e0 / M);
                    const long long r = e0 - (long long)k * M;
                    for (int c = 0; c < NE; ++c) test_cell<PT>(P, K, M, k, r + c, elem<PT>::val(P[e0 + c]), thr, peaks, capacity, count);
                }
            }
        }
    } else {
        for (long long e = tid; e < total; e += stride) {
            const int k = (int)(e / M);
            test_cell<PT>(P, K, M, k, e - (long long)k * M, elem<PT>::val(P[e]), thr, peaks, capacity, count);
        }
    }
}

// fdas_search, second kernel.  The convolve epilogue flagged (zi0, r): "one of the powers of bin
// r in |z| table entries zi0 .. zi0+span-1 exceeds the threshold".  Each thread takes one (entry,
// sign) of one candidate, reads that cell from the plane just written and applies the peak rule.
// If the candidate buffer overflowed, the whole plane is scanned instead (same result).
template <typename PT, typename VT, int NE>
__global__ void __launch_bounds__(256)
fdas_resolve_kernel(const PT *__restrict__ P, int K, long long M, float thr, const fdas_peak_t *__restrict__ cand,
                    const int *__restrict__ cand_count, int cand_capacity, int span, const int2 *__restrict__ ktab,
                    int nzg, fdas_peak_t *peaks, int capacity, int *count)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");   // launched as a programmatic dependent of the convolve launch
    const int n = *cand_count;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n <= cand_capacity) {
        const int cells = 2 * span;
        for (long long i = tid; i < (long long)cells * n; i += stride) {
            const fdas_peak_t c = cand[i / cells];
            const int zi = c.z_index + (int)((i % cells) >> 1);
            if (zi >= (c.z_index / nzg + 1) * nzg) continue;      // past the end of this template group
            const int2 kk = ktab[zi];
            const int k = (i & 1) ? kk.y : kk.x;
            if (k < 0 || ((i & 1) && kk.y == kk.x)) continue;      // no such row / z = 0 listed twice
            test_cell<PT>(P, K, M, k, c.r, elem<PT>::val(P[(size_t)k * M + c.r]), thr, peaks, capacity, count);
        }
        return;
    }
    const long long total = (long long)K * M;
    for (long long e = tid; e < total; e += stride) {
        const int k = (int)(e / M);
        test_cell<PT>(P, K, M, k, e - (long long)k * M, elem<PT>::val(P[e]), thr, peaks, capacity, count);
    }
}

// fdas_search on the overlap-save FFT forms: the convolve launch listed, per (thread, template), "one of my 16 outputs
// exceeds the threshold" (flag_outputs, fdas_convolve.cu: z_index = k, r = the thread's first output index i0 inside
// its segment, power = the bits of the segment number).  A record expands to the thread's outputs
// i = i0 + du(u) + 256 k3 (u < U = 16 / R3, k3 < R3 = S / 256; du = u for U <= 2, else (S / 16) u), of which those in
// the segment's valid window [L, L + V) and inside the plane are read back and tested.  Overflow of the list:
// whole-plane scan (same result).
template <typename PT>
__global__ void __launch_bounds__(256)
fdas_resolve_cells_kernel(const PT *__restrict__ P, int K, long long M, float thr, const fdas_peak_t *__restrict__ cand,
                          const int *__restrict__ cand_count, int cand_capacity, int S, int L, int V, fdas_peak_t *peaks,
                          int capacity, int *count)
{
    const int n = *cand_count;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (n <= cand_capacity) {
        const int R3 = S / 256, U = 16 / R3, T = S / 16;
        for (long long j = tid; j < 16LL * n; j += stride) {
            const fdas_peak_t c = cand[j >> 4];
            const int o = (int)(j & 15), u = o / R3, k3 = o % R3;
            const int i = c.r + (U <= 2 ? u : T * u) + 256 * k3;
            const long long col = (long long)__float_as_int(c.power) * V - L + i;
            if (i < L || i >= L + V || col >= M) continue;
            test_cell<PT>(P, K, M, c.z_index, col, elem<PT>::val(P[(size_t)c.z_index * M + col]), thr, peaks, capacity, count);
        }
        return;
    }
    const long long total = (long long)K * M;
    for (long long e = tid; e < total; e += stride) {
        const int k = (int)(e / M);
        test_cell<PT>(P, K, M, k, e - (long long)k * M, elem<PT>::val(P[e]), thr, peaks, capacity, count);
    }
}

// ---- f-fdot-fddot volume (fdas_volume_peaks; reading A27): the plane rule with one more axis.  V[i][k][r],
// i = 0..W-1; 26 neighbours, strictly greater than those that precede the cell in (i, k, r) order.
template <typename PT>
__device__ __forceinline__ void test_cell3(const PT *__restrict__ V, int W, int K, long long M, int i, int k, long long r,
                                           typename elem<PT>::cmp v, float thr, fdas_peak3_t *peaks, int capacity, int *count)
{
    using CT = typename elem<PT>::cmp;
    if (!(v > (CT)thr)) return;
    bool ok = true;
#pragma unroll
    for (int di = -1; di <= 1; ++di) {
#pragma unroll
        for (int dk = -1; dk <= 1; ++dk) {
#pragma unroll
            for (int dr = -1; dr <= 1; ++dr) {
                if (di == 0 && dk == 0 && dr == 0) continue;
                const int ii = i + di, kk = k + dk;
                const long long rr = r + dr;
                if (ii < 0 || ii >= W || kk < 0 || kk >= K || rr < 0 || rr >= M) continue;
                const CT n = elem<PT>::val(V[((size_t)ii * K + kk) * M + rr]);
                const bool precedes = (di < 0) || (di == 0 && (dk < 0 || (dk == 0 && dr < 0)));
                ok = ok && (precedes ? (v > n) : (v >= n));
            }
        }
    }
    if (ok) {
        const int slot = atomicAdd(count, 1);
        if (slot < capacity) {
            fdas_peak3_t rec;
            rec.w_index = i;
            rec.z_index = k;
            rec.r = (int32_t)r;
            rec.power = (float)v;
            peaks[slot] = rec;
        }
    }
}

template <typename PT, typename VT, int NE>
__global__ void __launch_bounds__(256)
fdas_peaks3_kernel(const PT *__restrict__ V, int W, int K, long long M, float thr, fdas_peak3_t *peaks, int capacity, int *count)
{
    const long long rows = (long long)W * K, total = rows * M;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (M % NE == 0) {
        const VT *PV = reinterpret_cast<const VT *>(V);
        const long long nv = total / NE;
        constexpr int UNR = 4;   // four 128-bit streaming loads in flight per thread (as fdas_peaks_kernel)
        for (long long q0 = tid; q0 < nv; q0 += UNR * stride) {
            union { VT v; PT e[NE]; } u[UNR];
#pragma unroll
            for (int j = 0; j < UNR; ++j)
                if (q0 + j * stride < nv) u[j].v = __ldcs(PV + q0 + j * stride);
#pragma unroll
            for (int j = 0; j < UNR; ++j) {
                const long long q = q0 + j * stride;
                if (q >= nv) break;
                using CT = typename elem<PT>::cmp;
                CT m = elem<PT>::val(u[j].e[0]);
#pragma unroll
                for (int c = 1; c < NE; ++c) m = max(m, elem<PT>::val(u[j].e[c]));
                if (m > (CT)thr) {
                    const long long e0 = q * NE;
                    const long long row = e0 / M;
                    const long long r = e0 - row * M;
                    const int i = (int)(row / K), k = (int)(row - (long long)i * K);
                    for (int c = 0; c < NE; ++c) test_cell3<PT>(V, W, K, M, i, k, r + c, elem<PT>::val(V[e0 + c]), thr, peaks, capacity, count);
                }
            }
        }
    } else {
        for (long long e = tid; e < total; e += stride) {
            const long long row = e / M;
            const int i = (int)(row / K), k = (int)(row - (long long)i * K);
            test_cell3<PT>(V, W, K, M, i, k, e - row * M, elem<PT>::val(V[e]), thr, peaks, capacity, count);
        }
    }
}

// fdas_volume_search on the tensor-core path: slab i's convolve launch flagged its candidates exactly as for
// fdas_search; each candidate cell is read back from the volume just written and tested against its 26 neighbours
// (slabs i - 1 and i + 1 are complete: every slab is convolved before the first slab is resolved).  If the slab's
// candidate buffer overflowed, the whole slab is scanned instead (same result).  Nothing re-reads the volume.
template <typename PT>
__global__ void __launch_bounds__(256)
fdas_resolve3_kernel(const PT *__restrict__ V, int W, int K, long long M, int slab, float thr, const fdas_peak_t *__restrict__ cand,
                     const int *__restrict__ cand_count, int cand_capacity, int span, const int2 *__restrict__ ktab, int nzg,
                     fdas_peak3_t *peaks, int capacity, int *count)
{
    const int n = *cand_count;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const PT *S = V + (size_t)slab * K * M;
    if (n <= cand_capacity) {
        const int cells = 2 * span;
        for (long long i = tid; i < (long long)cells * n; i += stride) {
            const fdas_peak_t c = cand[i / cells];
            const int zi = c.z_index + (int)((i % cells) >> 1);
            if (zi >= (c.z_index / nzg + 1) * nzg) continue;      // past the end of this template group
            const int2 kk = ktab[zi];
            const int k = (i & 1) ? kk.y : kk.x;
            if (k < 0 || ((i & 1) && kk.y == kk.x)) continue;      // no such row / z = 0 listed twice
            test_cell3<PT>(V, W, K, M, slab, k, c.r, elem<PT>::val(S[(size_t)k * M + c.r]), thr, peaks, capacity, count);
        }
        return;
    }
    const long long total = (long long)K * M;
    for (long long e = tid; e < total; e += stride) {
        const int k = (int)(e / M);
        test_cell3<PT>(V, W, K, M, slab, k, e - (long long)k * M, elem<PT>::val(S[e]), thr, peaks, capacity, count);
    }
}

}  // namespace

int fdas_launch_resolve_cells(fdas_plan *p, const void *plane, const fdas_search_args &sa, fdas_peak_t *peaks, int capacity, cudaStream_t st)
{
    const int grid = p->num_sms * 2;
    if (p->precision == FDAS_F64)
        fdas_resolve_cells_kernel<double><<<grid, 256, 0, st>>>((const double *)plane, p->K, p->M, sa.thr, sa.cand, sa.cand_count,
                                                                sa.cand_capacity, p->S, p->L, p->V, peaks, capacity, sa.count_out);
    else if (p->plane_bf16)
        fdas_resolve_cells_kernel<bf16raw><<<grid, 256, 0, st>>>((const bf16raw *)plane, p->K, p->M, sa.thr, sa.cand, sa.cand_count,
                                                                 sa.cand_capacity, p->S, p->L, p->V, peaks, capacity, sa.count_out);
    else
        fdas_resolve_cells_kernel<float><<<grid, 256, 0, st>>>((const float *)plane, p->K, p->M, sa.thr, sa.cand, sa.cand_count,
                                                               sa.cand_capacity, p->S, p->L, p->V, peaks, capacity, sa.count_out);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

int fdas_launch_resolve3(fdas_plan *p, const void *volume, int n_slabs, int slab, const fdas_search_args &sa, fdas_peak3_t *peaks,
                         int capacity, int *count, cudaStream_t st)
{
    const int grid = p->num_sms * 2;
    fdas_resolve3_kernel<float><<<grid, 256, 0, st>>>((const float *)volume, n_slabs, p->K, p->M, slab, sa.thr, sa.cand, sa.cand_count,
                                                      sa.cand_capacity, sa.cand_span, p->tc_ktab, p->tc_nzg, peaks, capacity, count);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

int fdas_launch_peaks3(fdas_plan *p, const void *volume, int n_slabs, float thr, fdas_peak3_t *peaks, int capacity, int *count,
                       cudaStream_t st)
{
    FDAS_CUDA_TRY(p, cudaMemsetAsync(count, 0, sizeof(int), st));
    const long long total = (long long)n_slabs * p->K * p->M;
    long long want = (total / 4 + 255) / 256;
    const long long cap = (long long)p->num_sms * 8;
    const int grid = (int)(want < cap ? (want > 0 ? want : 1) : cap);
    if (p->precision == FDAS_F64)
        fdas_peaks3_kernel<double, double2, 2><<<grid, 256, 0, st>>>((const double *)volume, n_slabs, p->K, p->M, thr, peaks, capacity, count);
    else if (p->plane_bf16)
        fdas_peaks3_kernel<bf16raw, uint4, 8><<<grid, 256, 0, st>>>((const bf16raw *)volume, n_slabs, p->K, p->M, thr, peaks, capacity, count);
    else
        fdas_peaks3_kernel<float, float4, 4><<<grid, 256, 0, st>>>((const float *)volume, n_slabs, p->K, p->M, thr, peaks, capacity, count);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    return FDAS_OK;
}

int fdas_launch_resolve(fdas_plan *p, const void *plane, const fdas_search_args &sa, fdas_peak_t *peaks, int capacity,
                        cudaStream_t st)
{
    // programmatic dependent launch: the grid is set up while the convolve launch drains; the kernel itself waits
    // (griddepcontrol.wait) for that launch to complete before it reads the candidates
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(p->num_sms * 2));
    cfg.blockDim = dim3(256);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (p->plane_bf16)
        FDAS_CUDA_TRY(p, cudaLaunchKernelEx(&cfg, fdas_resolve_kernel<bf16raw, uint4, 8>, (const bf16raw *)plane, p->K, (long long)p->M, sa.thr,
                                            (const fdas_peak_t *)sa.cand, (const int *)sa.cand_count, sa.cand_capacity, sa.cand_span,
                                            (const int2 *)p->tc_ktab, p->tc_nzg, peaks, capacity, sa.count_out));
    else
        FDAS_CUDA_TRY(p, cudaLaunchKernelEx(&cfg, fdas_resolve_kernel<float, float4, 4>, (const float *)plane, p->K, (long long)p->M, sa.thr,
                                            (const fdas_peak_t *)sa.cand, (const int *)sa.cand_count, sa.cand_capacity, sa.cand_span,
                                            (const int2 *)p->tc_ktab, p->tc_nzg, peaks, capacity, sa.count_out));
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

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
    else if (p->plane_bf16)
        fdas_peaks_kernel<bf16raw, uint4, 8><<<grid, 256, 0, st>>>((const bf16raw *)plane, p->K, p->M, thr, peaks, capacity, count);
    else
        fdas_peaks_kernel<float, float4, 4><<<grid, 256, 0, st>>>((const float *)plane, p->K, p->M, thr, peaks, capacity, count);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
