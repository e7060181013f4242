// fdas_convolve.cu -- the fused overlap-save convolution kernel (include/fdas.h: fdas_convolve).
//
// PAPER.md:65-67 (overlap-save: window the spectrum, convolve each window with every
// template by FFT, keep the central region) and PAPER.md:59 (the result is the f-fdot power
// plane).  In AstroAccelerate each arrow of Fig. 1 is a kernel or a library FFT with its
// intermediate in HBM ("limited by memory bandwidth"); here one CTA does the
// whole chain for one segment and a group of templates and only the V valid powers per
// (segment, template) ever reach HBM.
//
// Transform structure (S = 16 * 16 * R3, T = S/16 threads, 16 points per thread):
//   layout A : thread t, slot a  <-> index t + T a                     (input of a transform)
//   pass 1   : 16-point DFT over a, twiddle W_S^(t k1), exchange through shared memory
//   pass 2   : thread (k1, n3) = (t / R3, t % R3): 16-point DFT over n2, twiddle
//              W_(16 R3)^(n3 k2), exchange
//   pass 3   : R3-point DFTs; output index i = k1 + 16 k2 + 256 k3      (natural order)
// The forward transform of the segment runs once per CTA through the same passes (real and
// imaginary parts swapped) and is kept in registers (fp32) or shared memory (fp64) in layout
// A; the bank is stored in layout A as well, so the per-template work is
//   G = F * H_k  ->  pass 1..3  ->  |y|^2  ->  store bins [L, L+V).
#include <cuda_bf16.h>
#include <stdio.h>
#include "fdas_fft.cuh"
#include "fdas_internal.h"

namespace {

using namespace fdas;

// Register budgets and the template prefetch of the fp32 / bf16 kernels (measured on config 3)
#define FDAS_F32_PREFETCH 1
#define FDAS_F32_REGS 168
#define FDAS_BF16_REGS 128

struct ConvParams {
    const void *spectra;  // [batch][M] complex
    void *planes;         // [batch][K][M]
    const void *bank;     // kernel-native order
    const void *twiddle;  // [S] exp(+2 pi i j / S)
    long long M;
    long long n_seg;
    int K, L, V;
    int k_per_group;
    fdas_search_args search;   // fdas_search: the cells above the threshold are listed while they are stored (SEARCH kernels)
};

// ---- per-precision traits -------------------------------------------------------------
struct TraitsF64 {
    using CT = double;
    using CT2 = double2;
    using PT = double;        // plane element
    using E = double2;        // exchange element in shared memory
    static constexpr int VC = 1;              // complexes per 16-byte bank vector
    static constexpr bool F_IN_REGS = true;
    static constexpr bool TW_IN_REGS = false;
    static constexpr bool PREFETCH_H = false;
    static constexpr bool ROUND_INPUT = false;
    static constexpr int REG_TARGET = 255;
    static __device__ __forceinline__ E pack(CT re, CT im) { return make_double2(re, im); }
    static __device__ __forceinline__ void unpack(E v, CT &re, CT &im) { re = v.x; im = v.y; }
    static __device__ __forceinline__ void bank_unpack(const uint4 &v, CT *re, CT *im)
    {
        re[0] = __longlong_as_double(((long long)v.y << 32) | v.x);
        im[0] = __longlong_as_double(((long long)v.w << 32) | v.z);
    }
};

struct TraitsF32 {
    using CT = float;
    using CT2 = float2;
    using PT = float;
    using E = float2;
    static constexpr int VC = 2;
    static constexpr bool F_IN_REGS = true;
    static constexpr bool TW_IN_REGS = true;
    static constexpr bool PREFETCH_H = FDAS_F32_PREFETCH != 0;
    static constexpr bool ROUND_INPUT = false;
    static constexpr int REG_TARGET = FDAS_F32_REGS;
    static __device__ __forceinline__ E pack(CT re, CT im) { return make_float2(re, im); }
    static __device__ __forceinline__ void unpack(E v, CT &re, CT &im) { re = v.x; im = v.y; }
    static __device__ __forceinline__ void bank_unpack(const uint4 &v, CT *re, CT *im)
    {
        re[0] = __uint_as_float(v.x); im[0] = __uint_as_float(v.y);
        re[1] = __uint_as_float(v.z); im[1] = __uint_as_float(v.w);
    }
};

// bf16 storage / fp32 accumulate (reading A12): spectrum rounded on load, bf16
// bank, bf16 staging of every shared-memory exchange, fp32 arithmetic, fp32 plane.
struct TraitsBF16 {
    using CT = float;
    using CT2 = float2;
    using PT = float;
    using E = unsigned int;   // packed bf16x2: low half = re, high half = im
    static constexpr int VC = 4;
    static constexpr bool F_IN_REGS = true;
    static constexpr bool TW_IN_REGS = true;
    static constexpr bool PREFETCH_H = true;
    static constexpr bool ROUND_INPUT = true;
    static constexpr int REG_TARGET = FDAS_BF16_REGS;
    static __device__ __forceinline__ E pack(CT re, CT im)
    {
        __nv_bfloat162 v = __floats2bfloat162_rn(re, im);   // .x = re (low), .y = im (high)
        return *reinterpret_cast<unsigned int *>(&v);
    }
    static __device__ __forceinline__ void unpack(E v, CT &re, CT &im)
    {
        re = __uint_as_float(v << 16);
        im = __uint_as_float(v & 0xffff0000u);
    }
    static __device__ __forceinline__ void bank_unpack(const uint4 &v, CT *re, CT *im)
    {
        unpack(v.x, re[0], im[0]);
        unpack(v.y, re[1], im[1]);
        unpack(v.z, re[2], im[2]);
        unpack(v.w, re[3], im[3]);
    }
};

template <typename T> __device__ __forceinline__ T round_bf16(T x) { return x; }
template <> __device__ __forceinline__ float round_bf16<float>(float x)
{
    return __bfloat162float(__float2bfloat16_rn(x));
}

template <typename PT> __device__ __forceinline__ void store_stream(PT *p, PT v) { __stcs(p, v); }
__device__ __forceinline__ void store_stream2(float *p, float a, float b) { __stcs((float2 *)p, make_float2(a, b)); }
__device__ __forceinline__ void store_stream2(double *p, double a, double b) { __stcs((double2 *)p, make_double2(a, b)); }

template <class Tr, int S> struct Geo {
    static constexpr int T = S / 16;
    static constexpr int R3 = S / 256;
    static constexpr int U = 16 / R3;                       // radix-R3 butterflies per thread
    static constexpr int STR1 = T + R3;                     // exchange-1 row stride (elements)
    static constexpr int EPW = 128 / (int)sizeof(typename Tr::E);   // elements per 128-byte wavefront
    static constexpr int PAD2 = (EPW / R3) > 1 ? (EPW / R3) : 1;
    static constexpr int STR2 = 256 + PAD2;                 // exchange-2 row stride
    static constexpr int SM1 = 16 * STR1;                   // elements
    static constexpr int SM2 = R3 * STR2;
    static constexpr size_t XCH_BYTES = (size_t)(SM1 + SM2) * sizeof(typename Tr::E);
    static constexpr size_t NAT_BYTES = (size_t)S * sizeof(typename Tr::CT2);   // natural-order view
    static constexpr size_t XCH_REGION = XCH_BYTES > NAT_BYTES ? XCH_BYTES : NAT_BYTES;
    static constexpr size_t F_BYTES = Tr::F_IN_REGS ? 0 : NAT_BYTES;
    static constexpr size_t XCH_ALIGNED = ((XCH_REGION + 15) / 16) * 16;
    static constexpr size_t TW2_BYTES = (size_t)16 * R3 * sizeof(typename Tr::CT2);   // [k2][n3] table
    static constexpr size_t SMEM_BYTES = XCH_ALIGNED + F_BYTES + TW2_BYTES;
    // resident CTAs per SM the register budget allows at Tr::REG_TARGET registers per thread
    static constexpr int MIN_BLOCKS_RAW = 65536 / (T * Tr::REG_TARGET);
    static constexpr int MIN_BLOCKS = MIN_BLOCKS_RAW < 1 ? 1 : (MIN_BLOCKS_RAW > 16 ? 16 : MIN_BLOCKS_RAW);
    // pass-3 butterfly index handled by thread t, sub-index u
    static __device__ __forceinline__ int bfly(int t, int u) { return (U <= 2) ? U * t + u : t + T * u; }
};

// Passes 1 and 2 of the inverse-sign transform.  In: layout A registers.  Out: exchange-2
// buffer written and the CTA synchronised; pass 3 reads it.  Pass-1 twiddles W_S^(t k1) are
// per-thread constants (registers, or the global table in fp64); pass-2 twiddles
// W_(16 R3)^(n3 k2) come from a 16 x R3 shared-memory table (conflict-free: the R3 distinct
// entries a warp needs for one k2 are contiguous).
template <class Tr, int S, bool TWR>
__device__ __forceinline__ void passes12(typename Tr::CT *re, typename Tr::CT *im, typename Tr::E *sm1,
                                         typename Tr::E *sm2, const typename Tr::CT2 *__restrict__ tw,
                                         const typename Tr::CT *tw1r, const typename Tr::CT *tw1i,
                                         const typename Tr::CT2 *tw2, int t)
{
    using G = Geo<Tr, S>;
    using CT = typename Tr::CT;
    constexpr int R3 = G::R3;
    const int n3 = t % R3, k1p = t / R3;
    // ---- pass 1
    Dft<CT, 16>::run(re, im);
#pragma unroll
    for (int k1 = 0; k1 < 16; ++k1) {
        const int s = DftSlot<16>::of(k1);
        if (k1 > 0) {
            if constexpr (TWR) {
                cmul(re[s], im[s], tw1r[k1], tw1i[k1]);
            } else {
                const typename Tr::CT2 w = tw[t * k1];
                cmul(re[s], im[s], w.x, w.y);
            }
        }
        sm1[k1 * G::STR1 + t] = Tr::pack(re[s], im[s]);
    }
    __syncthreads();
    // ---- pass 2
#pragma unroll
    for (int n2 = 0; n2 < 16; ++n2) Tr::unpack(sm1[k1p * G::STR1 + n2 * R3 + n3], re[n2], im[n2]);
    Dft<CT, 16>::run(re, im);
#pragma unroll
    for (int k2 = 0; k2 < 16; ++k2) {
        const int s = DftSlot<16>::of(k2);
        if (k2 > 0 && R3 > 1) {
            const typename Tr::CT2 w = tw2[k2 * R3 + n3];
            cmul(re[s], im[s], w.x, w.y);
        }
        sm2[n3 * G::STR2 + k1p + 16 * k2] = Tr::pack(re[s], im[s]);
    }
    __syncthreads();
}

// Pass 3 for butterfly sub-index u: leaves y[b + 256 k3] in (re, im)[DftSlot<R3>::of(k3)].
template <class Tr, int S>
__device__ __forceinline__ void pass3(typename Tr::CT *re, typename Tr::CT *im, const typename Tr::E *sm2, int b)
{
    using G = Geo<Tr, S>;
#pragma unroll
    for (int n3 = 0; n3 < G::R3; ++n3) Tr::unpack(sm2[n3 * G::STR2 + b], re[n3], im[n3]);
    Dft<typename Tr::CT, G::R3>::run(re, im);
}

// fdas_search on the FFT forms: "one of the 16 outputs of thread i0's of segment `seg` for template k exceeds the
// threshold" -- one record per (thread, template), appended to the plan's candidate list; the resolve launch that
// follows expands it to the thread's valid cells and applies the peak rule to those (a few thousand of 4e8 cells on
// config 3).  The record reuses fdas_peak_t: z_index = k, r = i0 (the thread's first output index inside the
// segment), power = the bits of seg.
__device__ __noinline__ void flag_outputs(fdas_peak_t *cand, int *cand_count, int cand_capacity, int k, int i0, int seg)
{
    const int slot = atomicAdd(cand_count, 1);
    if (slot < cand_capacity) {
        fdas_peak_t rec;
        rec.z_index = k;
        rec.r = i0;
        rec.power = __int_as_float(seg);
        cand[slot] = rec;
    }
}

template <class Tr, int S, bool SEARCH = false>
__global__ void __launch_bounds__(S / 16, Geo<Tr, S>::MIN_BLOCKS) fdas_convolve_kernel(const ConvParams p)
{
    using G = Geo<Tr, S>;
    using CT = typename Tr::CT;
    using CT2 = typename Tr::CT2;
    using PT = typename Tr::PT;
    using E = typename Tr::E;
    constexpr int T = G::T, R3 = G::R3, U = G::U, VC = Tr::VC, NV = 16 / VC;
    constexpr bool TWR = Tr::TW_IN_REGS;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    E *sm1 = reinterpret_cast<E *>(smem_raw);
    E *sm2 = sm1 + G::SM1;
    CT2 *nat = reinterpret_cast<CT2 *>(smem_raw);  // natural-order view of the exchange region
    CT2 *smF = reinterpret_cast<CT2 *>(smem_raw + G::XCH_ALIGNED);

    const int t = threadIdx.x;
    if (SEARCH && t == 0 && blockIdx.x == 0 && blockIdx.y == 0) {
        *p.search.cand_count_next = 0;   // the other counter: nobody appends to it during this launch
        *p.search.count_out = 0;         // written by the resolve kernel that follows in stream order
    }
    const long long seg = blockIdx.x % p.n_seg;
    const long long ser = blockIdx.x / p.n_seg;
    const int k_begin = blockIdx.y * p.k_per_group;
    const int k_end = min(p.K, k_begin + p.k_per_group);
    const CT2 *__restrict__ tw = static_cast<const CT2 *>(p.twiddle);

    // twiddles that do not depend on the template
    CT2 *tw2 = reinterpret_cast<CT2 *>(smem_raw + G::XCH_ALIGNED + G::F_BYTES);
    for (int e = t; e < 16 * R3; e += T) tw2[e] = tw[16 * (e % R3) * (e / R3)];
    CT tw1r[TWR ? 16 : 1], tw1i[TWR ? 16 : 1];
    if constexpr (TWR) {
#pragma unroll
        for (int k = 1; k < 16; ++k) {
            const CT2 w = tw[t * k];
            tw1r[k] = w.x; tw1i[k] = w.y;
        }
    }
    // (the first __syncthreads inside passes12 orders the tw2 table writes before its reads)

    CT re[16], im[16];

    // ---- segment load (layout A), zero outside [0, M)   ("splitting the long
    //      input signal into windows")
    {
        const CT2 *__restrict__ X = static_cast<const CT2 *>(p.spectra) + ser * p.M;
        const long long g0 = seg * p.V - p.L + t;
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            const long long g = g0 + (long long)T * a;
            CT2 v;
            v.x = 0; v.y = 0;
            if (g >= 0 && g < p.M) v = X[g];
            if (Tr::ROUND_INPUT) { v.x = round_bf16(v.x); v.y = round_bf16(v.y); }
            // forward transform by the swap trick: feed (im, re)
            re[a] = v.y;
            im[a] = v.x;
        }
    }
    // ---- forward FFT, once per segment
    passes12<Tr, S, TWR>(re, im, sm1, sm2, tw, tw1r, tw1i, tw2, t);
    {
        CT2 fo[16];   // natural-order results of this thread: index bfly(t,u) + 256 k3
#pragma unroll
        for (int u = 0; u < U; ++u) {
            pass3<Tr, S>(re, im, sm2, G::bfly(t, u));
#pragma unroll
            for (int k3 = 0; k3 < R3; ++k3) {
                const int s = DftSlot<R3>::of(k3);
                fo[u * R3 + k3].x = im[s];   // un-swap
                fo[u * R3 + k3].y = re[s];
            }
        }
        __syncthreads();   // everyone is done reading sm2 before the natural-order view overwrites it
        CT2 *dstF = Tr::F_IN_REGS ? nat : smF;
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int k3 = 0; k3 < R3; ++k3) dstF[G::bfly(t, u) + 256 * k3] = fo[u * R3 + k3];
        __syncthreads();
    }
    CT Fr[Tr::F_IN_REGS ? 16 : 1], Fi[Tr::F_IN_REGS ? 16 : 1];
    if constexpr (Tr::F_IN_REGS) {
#pragma unroll
        for (int a = 0; a < 16; ++a) {
            const CT2 v = nat[t + T * a];
            Fr[a] = v.x; Fi[a] = v.y;
        }
        __syncthreads();   // nat aliases the exchange buffers
    }

    // ---- template loop
    const uint4 *__restrict__ bank = static_cast<const uint4 *>(p.bank);
    uint4 hv[Tr::PREFETCH_H ? NV : 1];
    if constexpr (Tr::PREFETCH_H) if (k_begin < k_end) {
#pragma unroll
        for (int v = 0; v < NV; ++v) hv[v] = __ldg(bank + ((size_t)k_begin * NV + v) * T + t);
    }
    // Output bookkeeping that does not depend on the template: which of this thread's 16
    // outputs (u, k3) -> i = bfly(t,u) + 256 k3 fall in the valid window [L, L+V) and inside
    // the plane ("discarding the contaminated regions at the edge of the windows").
    const long long col0 = seg * p.V - p.L;   // plane column of output index i is col0 + i
    const bool vec2 = (U == 2) && ((p.M & 1) == 0);
    unsigned vmask = 0;
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
        for (int k3 = 0; k3 < R3; ++k3) {
            const int i = G::bfly(t, u) + 256 * k3;
            if (i >= p.L && i < p.L + p.V && col0 + i < p.M) vmask |= 1u << (u * R3 + k3);
        }
    const long long out_off = (long long)ser * p.K * p.M + col0 + G::bfly(t, 0);   // + k*M per template
    PT *const plane = static_cast<PT *>(p.planes);

#pragma unroll 1
    for (int k = k_begin; k < k_end; ++k) {
        // G = F * H_k   (PAPER.md:35 convolution theorem)
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            uint4 h;
            if constexpr (Tr::PREFETCH_H) h = hv[v];
            else h = __ldg(bank + ((size_t)k * NV + v) * T + t);
            CT hr[VC], hi[VC];
            Tr::bank_unpack(h, hr, hi);
#pragma unroll
            for (int c = 0; c < VC; ++c) {
                const int a = v * VC + c;
                CT fr, fi;
                if constexpr (Tr::F_IN_REGS) { fr = Fr[a]; fi = Fi[a]; }
                else { const CT2 f = smF[t + T * a]; fr = f.x; fi = f.y; }
                re[a] = fr * hr[c] - fi * hi[c];
                im[a] = fr * hi[c] + fi * hr[c];
            }
        }
        if constexpr (Tr::PREFETCH_H) if (k + 1 < k_end) {
#pragma unroll
            for (int v = 0; v < NV; ++v) hv[v] = __ldg(bank + ((size_t)(k + 1) * NV + v) * T + t);
        }
        // inverse FFT
        passes12<Tr, S, TWR>(re, im, sm1, sm2, tw, tw1r, tw1i, tw2, t);
        PT *const row = plane + (out_off + (long long)k * p.M);   // &P[k][col0 + bfly(t,0)]
        if constexpr (U == 2) {
            CT pw[2][R3];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                pass3<Tr, S>(re, im, sm2, 2 * t + u);
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3) {
                    const int s = DftSlot<R3>::of(k3);
                    pw[u][k3] = re[s] * re[s] + im[s] * im[s];
                }
            }
            if constexpr (SEARCH && sizeof(CT) == 8) {
                // fp64: the largest power is tracked through the high words of the (non-negative) doubles, integer
                // maxima on the ALU pipe instead of 16 fp64 compares per template (the search variant cost 14 % more
                // than the plain one): hi(pw) >= hi(thr) holds whenever pw > thr, so the test is conservative and the
                // resolve launch, which tests every listed cell exactly, rejects the few extra records
                int hmx = -1;
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3) {
                    if (vmask & (1u << k3)) hmx = max(hmx, __double2hiint(pw[0][k3]));
                    if (vmask & (1u << (R3 + k3))) hmx = max(hmx, __double2hiint(pw[1][k3]));
                }
                if (hmx >= __double2hiint((double)p.search.thr) && hmx >= 0)
                    flag_outputs(p.search.cand, p.search.cand_count, p.search.cand_capacity, k, G::bfly(t, 0), (int)seg);
            } else if constexpr (SEARCH) {
                CT mx = 0;
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3) {
                    if (vmask & (1u << k3)) mx = max(mx, pw[0][k3]);
                    if (vmask & (1u << (R3 + k3))) mx = max(mx, pw[1][k3]);
                }
                if ((PT)mx > (PT)p.search.thr) flag_outputs(p.search.cand, p.search.cand_count, p.search.cand_capacity, k, G::bfly(t, 0), (int)seg);   // the stored value, compared in the plane's type as fdas_peaks does
            }
            if (vec2) {
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3)
                    if (vmask & (1u << k3)) store_stream2(row + 256 * k3, (PT)pw[0][k3], (PT)pw[1][k3]);
            } else {
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3) {
                    if (vmask & (1u << k3)) store_stream(row + 256 * k3, (PT)pw[0][k3]);
                    if (vmask & (1u << (R3 + k3))) store_stream(row + 256 * k3 + 1, (PT)pw[1][k3]);
                }
            }
        } else {
            PT mx_g = 0;
            int hmx_g = -1;   // fp64: high words, as above
#pragma unroll
            for (int u = 0; u < U; ++u) {
                pass3<Tr, S>(re, im, sm2, G::bfly(t, u));
#pragma unroll
                for (int k3 = 0; k3 < R3; ++k3) {
                    const int s = DftSlot<R3>::of(k3);
                    if (vmask & (1u << (u * R3 + k3))) {
                        const PT pv = (PT)(re[s] * re[s] + im[s] * im[s]);
                        store_stream(row + (G::bfly(t, u) - G::bfly(t, 0)) + 256 * k3, pv);
                        if constexpr (SEARCH && sizeof(PT) == 8) hmx_g = max(hmx_g, __double2hiint((double)pv));
                        else if constexpr (SEARCH) mx_g = max(mx_g, pv);
                    }
                }
            }
            if constexpr (SEARCH) {
                const bool hit = sizeof(PT) == 8 ? (hmx_g >= 0 && hmx_g >= __double2hiint((double)p.search.thr)) : (mx_g > (PT)p.search.thr);
                if (hit) flag_outputs(p.search.cand, p.search.cand_count, p.search.cand_capacity, k, G::bfly(t, 0), (int)seg);
            }
        }
        // no barrier needed here: the next template's first shared-memory write (exchange 1)
        // touches sm1, whose last readers finished before this template's second barrier;
        // sm2 is rewritten only after the next template's first barrier.
    }
}

template <class Tr, int S, bool SEARCH>
int launch_one(fdas_plan *p, const ConvParams &cp, int batch, int groups, cudaStream_t st)
{
    using G = Geo<Tr, S>;
    auto kern = fdas_convolve_kernel<Tr, S, SEARCH>;
    { const int rc = fdas_optin_smem(p, SEARCH ? FDAS_OPTIN_FFT_SEARCH : FDAS_OPTIN_FFT, kern, G::SMEM_BYTES); if (rc) return rc; }
    const long long gx = (long long)batch * p->n_seg;
    if (gx > 2147483647LL) return FDAS_ERR_INVALID_ARG;
    kern<<<dim3((unsigned)gx, groups), G::T, G::SMEM_BYTES, st>>>(cp);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}

// template groups of the FFT form: one forward FFT per (segment, group); the K templates are split only when there
// are too few segments to fill the GPU (e.g. config 1: 35 segments)
int fft_groups(const fdas_plan *p, int batch, int *k_per_group)
{
    const long long ctas = (long long)batch * p->n_seg;
    const long long want = 8LL * p->num_sms;
    int groups = 1;
    if (ctas < want) groups = (int)((want + ctas - 1) / ctas);
    if (groups > p->K) groups = p->K;
    *k_per_group = (p->K + groups - 1) / groups;
    return (p->K + *k_per_group - 1) / *k_per_group;
}

template <class Tr>
size_t smem_of(int S)
{
    switch (S) {
    case 256: return Geo<Tr, 256>::SMEM_BYTES;
    case 512: return Geo<Tr, 512>::SMEM_BYTES;
    case 1024: return Geo<Tr, 1024>::SMEM_BYTES;
    case 2048: return Geo<Tr, 2048>::SMEM_BYTES;
    case 4096: return Geo<Tr, 4096>::SMEM_BYTES;
    default: return 0;
    }
}

template <class Tr, bool SEARCH>
int launch_prec(fdas_plan *p, const ConvParams &cp, int batch, int groups, cudaStream_t st)
{
    switch (p->S) {
    case 256: return launch_one<Tr, 256, SEARCH>(p, cp, batch, groups, st);
    case 512: return launch_one<Tr, 512, SEARCH>(p, cp, batch, groups, st);
    case 1024: return launch_one<Tr, 1024, SEARCH>(p, cp, batch, groups, st);
    case 2048: return launch_one<Tr, 2048, SEARCH>(p, cp, batch, groups, st);
    case 4096: return launch_one<Tr, 4096, SEARCH>(p, cp, batch, groups, st);
    default: return FDAS_ERR_UNSUPPORTED;
    }
}

int launch_fft_form(fdas_plan *p, ConvParams &cp, int batch, const fdas_search_args *search, cudaStream_t st)
{
    const int groups = fft_groups(p, batch, &cp.k_per_group);
    cp.search = search ? *search : fdas_search_args{};
    if (search) {
        switch (p->precision) {
        case FDAS_F64: return launch_prec<TraitsF64, true>(p, cp, batch, groups, st);
        case FDAS_F32: return launch_prec<TraitsF32, true>(p, cp, batch, groups, st);
        case FDAS_BF16: return launch_prec<TraitsBF16, true>(p, cp, batch, groups, st);
        default: return FDAS_ERR_INVALID_ARG;
        }
    }
    switch (p->precision) {
    case FDAS_F64: return launch_prec<TraitsF64, false>(p, cp, batch, groups, st);
    case FDAS_F32: return launch_prec<TraitsF32, false>(p, cp, batch, groups, st);
    case FDAS_BF16: return launch_prec<TraitsBF16, false>(p, cp, batch, groups, st);
    default: return FDAS_ERR_INVALID_ARG;
    }
}

}  // namespace

int fdas_launch_convolve(fdas_plan *p, const void *spectra, void *planes, int batch, cudaStream_t st)
{
    if (fdas_uses_mma(p)) {
        const int rc = fdas_launch_convolve_mma(p, spectra, planes, batch, st);
        // fp32 under FDAS_ALGO_AUTO: a plane buffer the split-operand kernel cannot take goes to the FFT kernel
        if (!(rc == FDAS_ERR_UNSUPPORTED && p->precision == FDAS_F32 && p->algo == FDAS_ALGO_AUTO)) return rc;
    }
    ConvParams cp;
    cp.spectra = spectra;
    cp.planes = planes;
    cp.bank = p->bank;
    cp.twiddle = p->twiddle;
    cp.M = p->M;
    cp.n_seg = p->n_seg;
    cp.K = p->K;
    cp.L = p->L;
    cp.V = p->V;
    return launch_fft_form(p, cp, batch, nullptr, st);
}

// the overlap-save FFT form with the threshold test of fdas_search in its store loop (one series)
int fdas_launch_convolve_fft_search(fdas_plan *p, const void *spectrum, void *plane, const fdas_search_args *search, cudaStream_t st)
{
    ConvParams cp;
    cp.spectra = spectrum;
    cp.planes = plane;
    cp.bank = p->bank;
    cp.twiddle = p->twiddle;
    cp.M = p->M;
    cp.n_seg = p->n_seg;
    cp.K = p->K;
    cp.L = p->L;
    cp.V = p->V;
    return launch_fft_form(p, cp, 1, search, st);
}

int fdas_fft_describe(fdas_plan *p, int batch, fdas_kernel_info_t *out)
{
    int kpg = 0;
    const int groups = fft_groups(p, batch, &kpg);
    out->algorithm = FDAS_ALGO_FFT;
    out->split = 0;
    out->groups = groups;
    out->nch = 0;
    out->k_steps = 0;
    out->work_item_bins = p->V;
    out->grid_x = (int32_t)((long long)batch * p->n_seg);
    out->grid_y = groups;
    out->block_threads = p->S / 16;
    out->dynamic_smem_bytes = p->precision == FDAS_F64 ? smem_of<TraitsF64>(p->S) : p->precision == FDAS_F32 ? smem_of<TraitsF32>(p->S) : smem_of<TraitsBF16>(p->S);
    out->tensor_flops = 0.0;
    snprintf(out->kernel, sizeof(out->kernel), "fdas_convolve_kernel<%s, %d>",
             p->precision == FDAS_F64 ? "TraitsF64" : p->precision == FDAS_F32 ? "TraitsF32" : "TraitsBF16", p->S);
    return FDAS_OK;
}
