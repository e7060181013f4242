// fdas_rfft.cu -- the "Real FFT" ahead of the convolution (include/fdas.h: fdas_spectrum).
//
// PAPER.md:85 (Fig. 1): "The 'Real FFT' ... was intentionally left in single-precision as it does
// not significantly affect the overall execution time (it does not scale with K, the number of
// filters)".  X[k] = (1/sqrt N) sum_j x[j] exp(-2 pi i j k / N), k = 0..N/2-1 (readings A8,
// A9), computed in fp32 as a half-length complex FFT of z[m] = x[2m] + i x[2m+1] followed by the
// real-input unpacking; the half-length FFT (L = N/2 = L1 L2 points) is a four-step FFT:
//
//   pass A  L2/8 CTAs: 8 adjacent columns m2, FFT of length L1 over m1 in shared memory,
//           twiddle W_L^{m2 k1}, Y[k1 L2 + m2]                        (64-byte segments both ways)
//   pass B  L1/2 CTAs: 2 rows k1, FFT of length L2 over m2, Z[k1 + L1 k2]  (16-byte segments out)
//   pass C  X[k] = E + exp(-2 pi i k / N) O,  E = (Z[k] + conj Z[L-k]) / 2,  O = -i (Z[k] - conj Z[L-k]) / 2
//
// Three streaming passes over 8 L bytes: HBM-bound, and small beside one fdas_convolve.  The
// shared-memory FFT is a decimation-in-frequency with two radix-2 stages fused per barrier (natural
// in, bit-reversed out; the store un-reverses), twiddles from sincospif with exactly representable
// arguments.
#include <math.h>
#include "fdas_internal.h"

namespace {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// exp(-2 pi i num / den), den a power of two <= 2^24 and 0 <= num < 2^24: 2 num / den is exact in fp32
__device__ __forceinline__ float2 twiddle(unsigned num, unsigned den)
{
    float s, c;
    sincospif(-2.0f * (float)num / (float)den, &s, &c);
    return make_float2(c, s);
}

// In-place decimation-in-frequency FFTs of length n = 2^logn on `nbatch` sequences in shared memory:
// element i of sequence b sits at s[i * si + b * sb].  tw[j] = exp(-2 pi i j / n), j < n/2.  Two radix-2
// stages are fused in registers (one shared-memory round trip and one barrier per pair of stages);
// an odd logn ends with a single radix-2 stage.  Output bit-reversed.
template <bool BATCH_FASTEST>
__device__ __forceinline__ void smem_fft_dif(float2 *s, int logn, int nbatch, int si, int sb, const float2 *tw)
{
    const int n = 1 << logn;
    int lh = logn - 1;                                  // log2 of the current half size
    for (; lh >= 1; lh -= 2) {
        const int q = 1 << (lh - 1), nq = n >> 2;       // quarter of the current block; butterflies per sequence
        const int tstride = logn - 1 - lh;              // tw index shift for W_{4q}
        for (int e = threadIdx.x; e < nq * nbatch; e += blockDim.x) {
            int g, b;
            if (BATCH_FASTEST) {
                b = e % nbatch;
                g = e / nbatch;
            } else {
                g = e & (nq - 1);
                b = e >> (logn - 2);
            }
            const int j = g & (q - 1), base = ((g >> (lh - 1)) << (lh + 1)) + j;
            float2 *p0 = s + base * si + b * sb, *p1 = p0 + q * si, *p2 = p1 + q * si, *p3 = p2 + q * si;
            const float2 x0 = *p0, x1 = *p1, x2 = *p2, x3 = *p3;
            const float2 w1 = tw[j << tstride], w2 = tw[(2 * j) << tstride];
            const float2 u0 = make_float2(x0.x + x2.x, x0.y + x2.y), u1 = make_float2(x1.x + x3.x, x1.y + x3.y);
            const float2 u2 = cmul(make_float2(x0.x - x2.x, x0.y - x2.y), w1);
            const float2 d13 = make_float2(x1.x - x3.x, x1.y - x3.y);
            const float2 u3 = cmul(make_float2(d13.y, -d13.x), w1);      // (x1 - x3) W^{j+q} = (x1 - x3)(-i) W^j
            *p0 = make_float2(u0.x + u1.x, u0.y + u1.y);
            *p1 = cmul(make_float2(u0.x - u1.x, u0.y - u1.y), w2);
            *p2 = make_float2(u2.x + u3.x, u2.y + u3.y);
            *p3 = cmul(make_float2(u2.x - u3.x, u2.y - u3.y), w2);
        }
        __syncthreads();
    }
    if (lh == 0) {                                      // last radix-2 stage: neighbours, twiddle 1
        const int nb2 = n >> 1;
        for (int e = threadIdx.x; e < nb2 * nbatch; e += blockDim.x) {
            int g, b;
            if (BATCH_FASTEST) {
                b = e % nbatch;
                g = e / nbatch;
            } else {
                g = e & (nb2 - 1);
                b = e >> (logn - 1);
            }
            float2 *p0 = s + (2 * g) * si + b * sb, *p1 = p0 + si;
            const float2 a = *p0, c = *p1;
            *p0 = make_float2(a.x + c.x, a.y + c.y);
            *p1 = make_float2(a.x - c.x, a.y - c.y);
        }
        __syncthreads();
    }
}

__device__ __forceinline__ unsigned bitrev(unsigned v, int bits) { return bits ? __brev(v) >> (32 - bits) : 0u; }

constexpr int RF_CB = 8;      // columns per CTA in pass A (64-byte segments; 64 KB of shared memory -> 3 CTAs per SM)
constexpr int RF_RB = 2;      // rows per CTA in pass B
constexpr int RF_L2MAX = 12;  // log2 of the longest row FFT

// pass A: z viewed as [L1][L2]; this CTA takes columns m2 = 16 blockIdx.x .. +15
__global__ void __launch_bounds__(512) fdas_rfft_cols_kernel(const float2 *__restrict__ z, float2 *__restrict__ Y, int l1, int l2)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *s = reinterpret_cast<float2 *>(smem_raw);
    const int L1 = 1 << l1, L2 = 1 << l2;
    float2 *tw = s + L1 * RF_CB;
    const int m20 = blockIdx.x * RF_CB;
    for (int j = threadIdx.x; j < L1 / 2; j += blockDim.x) tw[j] = twiddle(j, L1);
    for (int e = threadIdx.x; e < L1 * RF_CB; e += blockDim.x) {
        const int m1 = e / RF_CB, c = e % RF_CB;
        s[e] = __ldg(z + (size_t)m1 * L2 + m20 + c);
    }
    __syncthreads();
    smem_fft_dif<true>(s, l1, RF_CB, RF_CB, 1, tw);
    for (int e = threadIdx.x; e < L1 * RF_CB; e += blockDim.x) {
        const int k1 = e / RF_CB, c = e % RF_CB;
        const float2 v = s[bitrev(k1, l1) * RF_CB + c];
        // four-step twiddle W_L^{m2 k1}: m2 k1 < 2^22
        Y[(size_t)k1 * L2 + m20 + c] = cmul(v, twiddle((unsigned)(m20 + c) * (unsigned)k1, 1u << (l1 + l2)));
    }
}

// pass B: rows k1 = 4 blockIdx.x .. +3 of Y [L1][L2] (or the single row when L1 == 1) -> Z[k1 + L1 k2]
__global__ void __launch_bounds__(512) fdas_rfft_rows_kernel(const float2 *__restrict__ Y, float2 *__restrict__ Z, int l1, int l2, int rb)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *s = reinterpret_cast<float2 *>(smem_raw);
    const int L1 = 1 << l1, L2 = 1 << l2;
    float2 *tw = s + L2 * rb;
    const int k10 = blockIdx.x * rb;
    for (int j = threadIdx.x; j < L2 / 2; j += blockDim.x) tw[j] = twiddle(j, L2);
    for (int e = threadIdx.x; e < L2 * rb; e += blockDim.x) s[e] = __ldg(Y + (size_t)k10 * L2 + e);   // rows are contiguous
    __syncthreads();
    smem_fft_dif<false>(s, l2, rb, 1, L2, tw);
    for (int e = threadIdx.x; e < L2 * rb; e += blockDim.x) {
        const int r = e % rb, k2 = e / rb;
        Z[(size_t)k2 * L1 + k10 + r] = s[r * L2 + bitrev(k2, l2)];
    }
}

// pass C: real-input unpacking, scale 1/sqrt(N); thread k handles bins k and L - k
template <typename OT2>
__global__ void __launch_bounds__(256) fdas_rfft_unpack_kernel(const float2 *__restrict__ Z, OT2 *__restrict__ X, unsigned L, float scale)
{
    for (unsigned k = blockIdx.x * blockDim.x + threadIdx.x; k <= L / 2; k += gridDim.x * blockDim.x) {
        const float2 a = Z[k], zb = Z[(L - k) & (L - 1)];
        const float2 b = make_float2(zb.x, -zb.y);
        const float2 E = make_float2(0.5f * (a.x + b.x), 0.5f * (a.y + b.y));
        const float2 d = make_float2(0.5f * (a.x - b.x), 0.5f * (a.y - b.y));
        const float2 O = make_float2(d.y, -d.x);                     // -i d
        float sn, cs;
        sincospif(-(float)k / (float)L, &sn, &cs);                   // exp(-2 pi i k / N), N = 2 L
        const float2 wO = cmul(make_float2(cs, sn), O);
        X[k].x = scale * (E.x + wO.x);
        X[k].y = scale * (E.y + wO.y);
        if (k != 0 && k != L - k) {                                  // X[L-k] = conj(E - w O)
            X[L - k].x = scale * (E.x - wO.x);
            X[L - k].y = -scale * (E.y - wO.y);
        }
    }
}

}  // namespace

int fdas_launch_spectrum(fdas_plan *p, const void *timeseries, void *spectrum, cudaStream_t st)
{
    int n = 0;
    while ((1LL << n) < p->N) ++n;
    if ((1LL << n) != p->N || n < 10 || n > 23) return FDAS_ERR_UNSUPPORTED;
    const int l = n - 1, l2 = l < RF_L2MAX ? l : RF_L2MAX, l1 = l - l2;
    const size_t L = (size_t)1 << l;
    if (!p->rfft_scratch) FDAS_CUDA_TRY(p, cudaMalloc(&p->rfft_scratch, 2 * L * sizeof(float2)));
    float2 *Y = static_cast<float2 *>(p->rfft_scratch), *Z = Y + L;
    const float2 *z = static_cast<const float2 *>(timeseries);
    if (l1 > 0) {
        const size_t smem = ((size_t)(1 << l1) * RF_CB + (1 << l1) / 2) * sizeof(float2);
        { const int rc = fdas_optin_smem(p, FDAS_OPTIN_RFFT_COLS, fdas_rfft_cols_kernel, smem); if (rc) return rc; }
        fdas_rfft_cols_kernel<<<(1 << l2) / RF_CB, 512, smem, st>>>(z, Y, l1, l2);
        FDAS_CUDA_TRY(p, cudaGetLastError());
        p->launches += 1;
    }
    {
        const int rb = l1 >= 2 ? RF_RB : 1;
        const size_t smem = ((size_t)(1 << l2) * rb + (1 << l2) / 2) * sizeof(float2);
        { const int rc = fdas_optin_smem(p, FDAS_OPTIN_RFFT_ROWS, fdas_rfft_rows_kernel, smem); if (rc) return rc; }
        fdas_rfft_rows_kernel<<<(1 << l1) / rb, 512, smem, st>>>(l1 > 0 ? Y : z, Z, l1, l2, rb);
        FDAS_CUDA_TRY(p, cudaGetLastError());
        p->launches += 1;
    }
    const float scale = (float)(1.0 / sqrt((double)p->N));
    const unsigned blocks = (unsigned)((L / 2 + 256) / 256 < (size_t)p->num_sms * 8 ? (L / 2 + 256) / 256 : (size_t)p->num_sms * 8);
    if (p->precision == FDAS_F64)
        fdas_rfft_unpack_kernel<double2><<<blocks, 256, 0, st>>>(Z, static_cast<double2 *>(spectrum), (unsigned)L, scale);
    else
        fdas_rfft_unpack_kernel<float2><<<blocks, 256, 0, st>>>(Z, static_cast<float2 *>(spectrum), (unsigned)L, scale);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
