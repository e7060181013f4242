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
// N >= 2^17 (both factors >= 256): passes A and B run the transforms in REGISTERS -- 16 points per thread, three
// butterfly passes of radix 16 / 16 / n/256 (the butterflies of fdas_fft.cuh), two shared-memory exchanges, output in
// natural order (fdas_rfft_fast_kernel below) -- and pass C is fused into pass B (a CTA takes rows and their mirror
// rows): two launches, the series read once, Y (8 L bytes, L2-resident) written and read once, the spectrum written once.  Smaller N keep the
// shared-memory decimation-in-frequency kernels (two radix-2 stages fused per barrier; natural in, bit-reversed
// out; the store un-reverses).  Twiddles come from sincospif with exactly representable arguments.
#include <math.h>
#include "fdas_fft.cuh"
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
constexpr int RF_NSEQ = 4;    // register FFT passes: adjacent columns / rows per CTA (32-byte segments; 8 needs 1024 threads at n = 2048)

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


// ---- register FFT passes (N >= 2^17) ---------------------------------------------------------------
// One length-n transform, n = 256 R3 (R3 = 1, 2, 4, 8, 16), by T = n / 16 threads holding 16 points each:
//   pass 1  thread t, slot a <-> input index t + T a: 16-point DFT over a -> k1; twiddle W_n^{t k1}
//   pass 2  thread (k1, t2), slot b <-> t = t2 + (T/16) b: 16-point DFT over b -> k2; twiddle W_T^{t2 k2}
//   pass 3  thread (k1, k2): R3-point DFTs over the remaining index (16 / R3 of them) -> k3
// output index k1 + 16 k2 + 256 k3: natural order, consecutive threads hold consecutive outputs.
// The butterflies are inverse-sign (exp(+2 pi i ..)); the forward transform is taken on data with re and im
// swapped and swapped back at the end (fdas_fft.cuh).  Sequences are interleaved by NSEQ in shared memory and in
// the thread index (sequence fastest) so that pass A reads / writes NSEQ adjacent columns (64-byte segments).
template <int R3>
struct FastGeo {
    static constexpr int N = 256 * R3, T = N / 16, U = 16 / R3;   // U radix-R3 butterflies per thread in pass 3
    static constexpr int STR1 = T + 1;                            // exchange 1: row k1 holds y_k1[t], padded
    static constexpr int STR2 = R3 + 2;                           // exchange 2: row (k2, k1) holds the R3 values t2, padded
    static constexpr int NEED = 16 * STR1 > 256 * STR2 ? 16 * STR1 : 256 * STR2;
    // elements per sequence, = 4 (mod 16): the sequences of a warp (8 of them x 4 consecutive t) then fall into
    // different 8-byte slots of a 128-byte wavefront
    static constexpr int SE = (NEED + 11) / 16 * 16 + 4;
};

// One transform per `seq`; re[], im[] hold the 16 inputs t + T a of thread t on entry and the outputs on exit:
// output index (t + T u) + 256 k3 sits in slot u R3 + DftSlot<R3>::of(k3).  tw[j] = exp(+2 pi i j / n), j < n.
template <int R3>
__device__ __forceinline__ void fast_fft(float *re, float *im, float2 *sx, const float2 *tw, int t, int seq)
{
    using G = FastGeo<R3>;
    using namespace fdas;
    constexpr int T = G::T, N = G::N;
    float2 *s1 = sx + (size_t)seq * G::SE;
    // pass 1: DFT16 over a; y_k1[t] = W_n^{t k1} sum_a x[t + T a] W_16^{a k1}
    Dft<float, 16>::run(re, im);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const int sl = DftSlot<16>::of(k1);
        float xr = re[sl], xi = im[sl];
        if (k1) {
            const float2 w = tw[(t * k1) & (N - 1)];
            fdas::cmul(xr, xi, w.x, w.y);
        }
        s1[k1 * G::STR1 + t] = make_float2(xr, xi);
    }
    __syncthreads();
    // pass 2: thread (k1, t2), t2 < R3: DFT16 over b of y_k1[t2 + R3 b]; twiddle W_T^{t2 k2} = W_n^{16 t2 k2}
    const int k1 = t / R3, t2 = t % R3;
#pragma unroll
    for (int b = 0; b < 16; ++b) {
        const float2 v = s1[k1 * G::STR1 + t2 + R3 * b];
        re[b] = v.x;
        im[b] = v.y;
    }
    __syncthreads();
    Dft<float, 16>::run(re, im);
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) {
        const int sl = DftSlot<16>::of(k2);
        float xr = re[sl], xi = im[sl];
        if (k2 && R3 > 1) {
            const float2 w = tw[(t2 * k2 * 16) & (N - 1)];
            fdas::cmul(xr, xi, w.x, w.y);
        }
        s1[(k2 * 16 + k1) * G::STR2 + t2] = make_float2(xr, xi);
    }
    __syncthreads();
    // pass 3: rows q = t + T u (q = k1 + 16 k2), R3-point DFT over t2 -> k3
#pragma unroll
    for (int u = 0; u < G::U; ++u) {
        const int row = t + T * u;
        const int rk1 = row & 15, rk2 = row >> 4;
#pragma unroll
        for (int j = 0; j < R3; ++j) {
            const float2 v = s1[(rk2 * 16 + rk1) * G::STR2 + j];
            re[u * R3 + j] = v.x;
            im[u * R3 + j] = v.y;
        }
        Dft<float, R3>::run(re + u * R3, im + u * R3);
    }
}

// Pass A (COLS = true): z viewed as [L1][L2]; CTA = NSEQ adjacent columns m2, transform over m1 (stride L2), output
// Y[k L2 + m2] = W_L^{m2 k} FFT_m1(z)[k].  Pass B (COLS = false): CTA = NSEQ rows k1 of Y [L1][L2] (contiguous),
// transform over m2; Z[k1 + L1 k2] never goes to memory: pass C (the real-input unpacking, file header) is done here.
// Bin k = k1 + L1 k2 needs Z[L - k], which sits in row L1 - k1 at k2' = L2 - 1 - k2 (rows 0 and L1/2 mirror onto
// themselves, row 0 at k2' = (L2 - k2) mod L2), so a CTA takes two rows and their two mirror rows -- rows
// 2b+1, 2b+2, L1-2b-1, L1-2b-2, the last CTA rows L1/2-1, L1/2+1, 0, L1/2 -- and the four transforms meet in shared memory.
template <int R3, bool COLS, int NSEQ, typename OT2>
__global__ void __launch_bounds__(FastGeo<R3>::T * NSEQ)
fdas_rfft_fast_kernel(const float2 *__restrict__ in, void *__restrict__ out_, int l1, int l2, float scale)
{
    using G = FastGeo<R3>;
    using namespace fdas;
    static_assert(COLS || NSEQ == 4, "pass B pairs two rows with their two mirror rows");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tw = reinterpret_cast<float2 *>(smem_raw);
    float2 *sx = tw + G::N;
    const int L2 = 1 << l2, L1 = 1 << l1;
    const int seq = threadIdx.x % NSEQ, t = threadIdx.x / NSEQ;
    for (int j = threadIdx.x; j < G::N; j += blockDim.x) {
        float sn, cs;
        sincospif(2.0f * (float)j / (float)G::N, &sn, &cs);
        tw[j] = make_float2(cs, sn);
    }
    float re[16], im[16];
    int k1 = 0, mate = seq;          // pass B: this thread's row; the sequence of this CTA that holds the mirror row
    if (COLS) {
        const int m2 = blockIdx.x * NSEQ + seq;
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            const float2 v = __ldg(in + (size_t)(t + G::T * a) * L2 + m2);
            re[a] = v.y;   // swapped: forward transform through the inverse-sign butterflies
            im[a] = v.x;
        }
    } else {
        // launched as a programmatic dependent of the column pass: the twiddle table above is built while that pass drains
        asm volatile("griddepcontrol.wait;" ::: "memory");
        const int b = blockIdx.x;
        if (b + 1 < (int)gridDim.x) {
            k1 = seq < 2 ? 2 * b + 1 + seq : L1 - 2 * b - 1 - (seq - 2);
            mate = seq ^ 2;
        } else {
            k1 = seq == 0 ? L1 / 2 - 1 : seq == 1 ? L1 / 2 + 1 : seq == 2 ? 0 : L1 / 2;
            mate = seq < 2 ? seq ^ 1 : seq;
        }
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            const float2 v = __ldg(in + (size_t)k1 * L2 + t + G::T * a);
            re[a] = v.y;
            im[a] = v.x;
        }
    }
    __syncthreads();   // twiddle table
    fast_fft<R3>(re, im, sx, tw, t, seq);
    constexpr int U = G::U;
    if (COLS) {
        // four-step twiddle W_L^{m2 k} = exp(-2 pi i m2 k / L), k = t + T (u + U k3): one sincospif per thread for
        // W_L^{m2 t} and a table of the 16 factors W_L^{m2 T j}, j = u + U k3, per sequence (arguments m2 k < 2^24:
        // 2 m2 k / L is exact in fp32, each factor is correctly rounded; their product adds one rounding, ~6e-8)
        float2 *out = static_cast<float2 *>(out_);
        const int m2 = blockIdx.x * NSEQ + seq;
        const float inv_L = 1.0f / (float)(1u << (l1 + l2));
        float2 *fac = sx + (size_t)NSEQ * G::SE;          // [NSEQ][16], behind the exchange buffers
        __syncthreads();
        if (t < 16) {
            float sn, cs;
            sincospif(-2.0f * (float)((unsigned)m2 * (unsigned)(G::T * t)) * inv_L, &sn, &cs);
            fac[seq * 16 + t] = make_float2(cs, sn);
        }
        float wsn, wcs;
        sincospif(-2.0f * (float)((unsigned)m2 * (unsigned)t) * inv_L, &wsn, &wcs);
        __syncthreads();
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int k3 = 0; k3 < R3; ++k3) {
                const int sl = u * R3 + DftSlot<R3>::of(k3);
                const int k = t + G::T * u + 256 * k3;
                float xr = im[sl], xi = re[sl];            // swap back: forward transform
                const float2 f = fac[seq * 16 + u + U * k3];
                float cs = wcs, sn = wsn;
                fdas::cmul(cs, sn, f.x, f.y);
                fdas::cmul(xr, xi, cs, sn);
                out[(size_t)k * L2 + m2] = make_float2(xr, xi);
            }
        }
    } else {
        // Z rows of this CTA -> shared memory (the exchange buffers are free after the barrier), natural k2 order
        OT2 *X = static_cast<OT2 *>(out_);
        float2 *zrow = sx + (size_t)seq * G::SE;
        __syncthreads();
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int k3 = 0; k3 < R3; ++k3) {
                const int sl = u * R3 + DftSlot<R3>::of(k3);
                zrow[t + G::T * u + 256 * k3] = make_float2(im[sl], re[sl]);   // swap back: forward transform
            }
        }
        __syncthreads();
        // pass C: X[k] = (E + exp(-2 pi i k / N) O) / sqrt N, E = (Z[k] + conj Z[L-k]) / 2, O = -i (Z[k] - conj Z[L-k]) / 2
        const float2 *zmate = sx + (size_t)mate * G::SE;
        const float inv_L = 1.0f / (float)(1u << (l1 + l2));
        // exp(-2 pi i k / N) = exp(-i pi (k1 + L1 t) / L) (one sincospif per thread) x exp(-i pi T j / L2), j = u + U k3
        float wsn, wcs;
        sincospif(-(float)((unsigned)k1 + ((unsigned)t << l1)) * inv_L, &wsn, &wcs);
#pragma unroll
        for (int u = 0; u < U; ++u) {
#pragma unroll
            for (int k3 = 0; k3 < R3; ++k3) {
                const int sl = u * R3 + DftSlot<R3>::of(k3);
                const int k2 = t + G::T * u + 256 * k3;
                const int k2m = k1 == 0 ? (L2 - k2) & (L2 - 1) : L2 - 1 - k2;
                const float2 a = make_float2(im[sl], re[sl]), zb = zmate[k2m];
                const float2 bq = make_float2(zb.x, -zb.y);
                const float2 E = make_float2(0.5f * (a.x + bq.x), 0.5f * (a.y + bq.y));
                const float2 d = make_float2(0.5f * (a.x - bq.x), 0.5f * (a.y - bq.y));
                const float2 O = make_float2(d.y, -d.x);                     // -i d
                const unsigned k = (unsigned)k1 + ((unsigned)k2 << l1);
                const float2 f = tw[(G::T / 2) * (u + U * k3)];             // exp(+i pi T j / L2): conjugate it
                const float2 wO = cmul(cmul(make_float2(wcs, wsn), make_float2(f.x, -f.y)), O);
                X[k].x = scale * (E.x + wO.x);
                X[k].y = scale * (E.y + wO.y);
            }
        }
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

template <int R3, bool COLS, typename OT2>
int launch_fast_r(fdas_plan *p, int l1, int l2, const float2 *in, void *out, float scale, cudaStream_t st)
{
    using G = FastGeo<R3>;
    constexpr int NSEQ = RF_NSEQ;
    auto kern = fdas_rfft_fast_kernel<R3, COLS, NSEQ, OT2>;
    const size_t smem = ((size_t)G::N + (size_t)NSEQ * G::SE + (size_t)NSEQ * 16) * sizeof(float2);
    { const int rc = fdas_optin_smem(p, (COLS ? FDAS_OPTIN_RFFT_COLS : sizeof(OT2) == 16 ? FDAS_OPTIN_RFFT_ROWS64 : FDAS_OPTIN_RFFT_ROWS), kern, smem); if (rc) return rc; }
    const int seqs = COLS ? (1 << l2) : (1 << l1);       // columns m2 / rows k1
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(seqs / NSEQ);
    cfg.blockDim = dim3(G::T * NSEQ);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // row pass: set up while the column pass drains
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = COLS ? 0 : 1;
    FDAS_CUDA_TRY(p, cudaLaunchKernelEx(&cfg, kern, in, out, l1, l2, scale));
    p->launches += 1;
    return FDAS_OK;
}

// pass A: transforms of length 2^l1 down the columns of [L1][L2]
int launch_fast_cols(fdas_plan *p, int l1, int l2, const float2 *in, float2 *out, cudaStream_t st)
{
    switch (l1 - 8) {
    case 0: return launch_fast_r<1, true, float2>(p, l1, l2, in, out, 1.f, st);
    case 1: return launch_fast_r<2, true, float2>(p, l1, l2, in, out, 1.f, st);
    case 2: return launch_fast_r<4, true, float2>(p, l1, l2, in, out, 1.f, st);
    case 3: return launch_fast_r<8, true, float2>(p, l1, l2, in, out, 1.f, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}
// pass B + C: transforms of length 2^l2 along the rows, unpacked and scaled into the spectrum
template <typename OT2>
int launch_fast_rows(fdas_plan *p, int l1, int l2, const float2 *in, void *spectrum, float scale, cudaStream_t st)
{
    switch (l2 - 8) {
    case 0: return launch_fast_r<1, false, OT2>(p, l1, l2, in, spectrum, scale, st);
    case 1: return launch_fast_r<2, false, OT2>(p, l1, l2, in, spectrum, scale, st);
    case 2: return launch_fast_r<4, false, OT2>(p, l1, l2, in, spectrum, scale, st);
    case 3: return launch_fast_r<8, false, OT2>(p, l1, l2, in, spectrum, scale, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}

}  // namespace

int fdas_launch_spectrum(fdas_plan *p, const void *timeseries, void *spectrum, cudaStream_t st)
{
    int n = 0;
    while ((1LL << n) < p->N) ++n;
    if ((1LL << n) != p->N || n < 10 || n > 23) return FDAS_ERR_UNSUPPORTED;
    const int l = n - 1;
    const size_t L = (size_t)1 << l;
    if (!p->rfft_scratch) FDAS_CUDA_TRY(p, cudaMalloc(&p->rfft_scratch, 2 * L * sizeof(float2)));
    float2 *Y = static_cast<float2 *>(p->rfft_scratch), *Z = Y + L;
    const float2 *z = static_cast<const float2 *>(timeseries);
    if (l >= 16) {
        // register FFT passes: L = L1 L2 with both factors in 256 .. 2048
        const int l1 = (l + 1) / 2, l2 = l - l1;
        const float scale = (float)(1.0 / sqrt((double)p->N));
        int rc = launch_fast_cols(p, l1, l2, z, Y, st);
        if (rc == FDAS_OK)
            rc = p->precision == FDAS_F64 ? launch_fast_rows<double2>(p, l1, l2, Y, spectrum, scale, st)
                                          : launch_fast_rows<float2>(p, l1, l2, Y, spectrum, scale, st);
        return rc;
    } else {
        const int l2 = l < RF_L2MAX ? l : RF_L2MAX, l1 = l - l2;
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
