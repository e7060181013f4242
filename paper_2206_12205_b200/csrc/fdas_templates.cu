// fdas_templates.cu -- template builder (include/fdas.h: fdas_build_templates).
//
// PAPER.md:37 / :105: each template is the Fourier response of a constant-fdot signal
// (Ransom et al. 2002), "a 1D array of complex numbers".  The paper generates it in fp32
// and converts; this build evaluates in fp64 and rounds once (reading A11).
//
//   taps kernel : h_z[j] = conj( int_0^1 exp(2 pi i [ j u + (z/2)(u^2-u) ]) du ),
//                 128 panels x 16-point Gauss-Legendre per tap, phase reduced modulo one
//                 cycle with error-free products so the taps are good to ~1e-16.
//   bank kernel : H_z[f] = (1/S) sum_j h_z[j] exp(-2 pi i f j / S) as a direct DFT over the
//                 2 m_z + 1 non-zero taps (exact integer angle reduction), rounded to the
//                 storage type and written in the convolve kernel's native order.
//   twiddles    : exp(+2 pi i j / S), j < S, in the compute type.
#include <cuda_bf16.h>
#include <math.h>
#include "fdas_internal.h"

namespace {

constexpr int GL_N = 16;       // nodes per panel
constexpr int GL_PANELS = 128; // panels on [0,1]; one thread each

struct GaussLegendre {
    double d[GL_N];  // (x_i + 1) / (2 * GL_PANELS): offset of node i inside a panel
    double w[GL_N];  // w_i / (2 * GL_PANELS)
};

// Host: nodes/weights of the 16-point rule by Newton iteration on P_16 (long double).
GaussLegendre make_rule()
{
    GaussLegendre g;
    const int n = GL_N;
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int i = 0; i < n; ++i) {
        long double x = cosl(pi * (i + 0.75L) / (n + 0.5L)), pp = 1.0L;
        for (int it = 0; it < 64; ++it) {
            long double p1 = 1.0L, p2 = 0.0L;
            for (int k = 1; k <= n; ++k) {
                long double p3 = p2;
                p2 = p1;
                p1 = ((2.0L * k - 1.0L) * x * p2 - (k - 1.0L) * p3) / k;
            }
            pp = n * (x * p1 - p2) / (x * x - 1.0L);
            long double dx = p1 / pp;
            x -= dx;
            if (fabsl(dx) < 1e-20L) {
                // refresh the derivative at the converged root
                p1 = 1.0L, p2 = 0.0L;
                for (int k = 1; k <= n; ++k) {
                    long double p3 = p2;
                    p2 = p1;
                    p1 = ((2.0L * k - 1.0L) * x * p2 - (k - 1.0L) * p3) / k;
                }
                pp = n * (x * p1 - p2) / (x * x - 1.0L);
                break;
            }
        }
        g.d[i] = (double)((x + 1.0L) / (2.0L * GL_PANELS));
        g.w[i] = (double)(2.0L / ((1.0L - x * x) * pp * pp) / (2.0L * GL_PANELS));
    }
    return g;
}

// fractional part of a*b computed without losing the low bits of the product
__device__ __forceinline__ double frac_of_product(double a, double b)
{
    double p = a * b;
    double e = fma(a, b, -p);
    return (p - rint(p)) + e;
}

// grid (2*m_max+1, K), block GL_PANELS
__global__ void __launch_bounds__(GL_PANELS)
fdas_taps_kernel(double2 *taps, int K, int m_max, double zmax, double dz, double jerk, GaussLegendre rule)
{
    const int k = blockIdx.y;
    const int j = (int)blockIdx.x - m_max;
    const double z = -zmax + k * dz;
    const int m = (int)ceil(fabs(z) / 2.0 + fabs(jerk) / 12.0) + 16;
    __shared__ double sr[GL_PANELS], si[GL_PANELS];
    double accr = 0.0, acci = 0.0;
    if (abs(j) <= m) {
        const double a = (double)threadIdx.x / GL_PANELS;  // exact
        const double zh = 0.5 * z;
        const double q0 = a * a - a;                        // exact (a has 7 bits)
        const double base = frac_of_product((double)j, a) + frac_of_product(zh, q0);
        const double lin = 2.0 * a - 1.0;
#pragma unroll
        for (int i = 0; i < GL_N; ++i) {
            const double d = rule.d[i];
            // phase in cycles: j u + (z/2)(u^2 - u), u = a + d
            double cyc = base + ((double)j * d + zh * (d * lin + d * d));
            if (jerk != 0.0) {   // jerk slab (reading A25): + (w/12)(2u^3 - 3u^2 + u), u = a + d
                const double u = a + d;
                cyc += (jerk / 12.0) * (u * (u * (2.0 * u - 3.0) + 1.0));
            }
            double s, c;
            sincospi(2.0 * cyc, &s, &c);
            accr += rule.w[i] * c;
            acci += rule.w[i] * s;
        }
    }
    sr[threadIdx.x] = accr;
    si[threadIdx.x] = acci;
    __syncthreads();
    for (int h = GL_PANELS / 2; h > 0; h >>= 1) {
        if (threadIdx.x < h) {
            sr[threadIdx.x] += sr[threadIdx.x + h];
            si[threadIdx.x] += si[threadIdx.x + h];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0)
        taps[(size_t)k * (2 * m_max + 1) + blockIdx.x] = make_double2(sr[0], -si[0]);  // conj
}

template <typename ST> struct StoreComplex;
template <> struct StoreComplex<double> {
    static __device__ void put(void *bank, size_t off, double re, double im)
    {
        ((double2 *)bank)[off] = make_double2(re, im);
    }
};
template <> struct StoreComplex<float> {
    static __device__ void put(void *bank, size_t off, double re, double im)
    {
        ((float2 *)bank)[off] = make_float2((float)re, (float)im);
    }
};
template <> struct StoreComplex<__nv_bfloat16> {
    static __device__ void put(void *bank, size_t off, double re, double im)
    {
        __nv_bfloat162 v;
        v.x = __double2bfloat16(re);  // round-to-nearest-even, once, from fp64
        v.y = __double2bfloat16(im);
        ((__nv_bfloat162 *)bank)[off] = v;
    }
};

// grid (S/256, K), block 256: one thread per (k, f)
template <typename ST>
__global__ void __launch_bounds__(256)
fdas_bank_kernel(void *bank, const double2 *__restrict__ taps, int K, int S, int T, int VC, int m_max,
                 double zmax, double dz, double jerk)
{
    const int k = blockIdx.y;
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f >= S) return;
    const double z = -zmax + k * dz;
    const int m = (int)ceil(fabs(z) / 2.0 + fabs(jerk) / 12.0) + 16;
    const double2 *h = taps + (size_t)k * (2 * m_max + 1) + m_max;
    double accr = 0.0, acci = 0.0;
    const double inv = 2.0 / S;
    for (int j = -m; j <= m; ++j) {
        int e = (int)(((long long)f * j) % S);
        if (e < 0) e += S;
        double s, c;
        sincospi(inv * e, &s, &c);  // angle 2 pi e / S
        const double2 t = h[j];
        // t * exp(-i theta)
        accr += t.x * c + t.y * s;
        acci += t.y * c - t.x * s;
    }
    const double sc = 1.0 / S;
    StoreComplex<ST>::put(bank, fdas_bank_offset(k, f, T, VC), accr * sc, acci * sc);
}

template <typename CT2>
__global__ void fdas_twiddle_kernel(CT2 *tw, int S)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= S) return;
    double s, c;
    sincospi(2.0 * j / S, &s, &c);
    tw[j].x = c;
    tw[j].y = s;
}

}  // namespace

int fdas_launch_build_templates(fdas_plan *p, cudaStream_t st)
{
    static const GaussLegendre rule = make_rule();
    const int ntap = 2 * p->m_max + 1;
    fdas_taps_kernel<<<dim3(ntap, p->K), GL_PANELS, 0, st>>>(p->taps, p->K, p->m_max, p->zmax, p->dz, p->jerk, rule);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    const dim3 grid((p->S + 255) / 256, p->K);
    const int VC = fdas_bank_vc(p->precision);
    if (p->precision == FDAS_F64) {
        fdas_bank_kernel<double><<<grid, 256, 0, st>>>(p->bank, p->taps, p->K, p->S, p->T, VC, p->m_max, p->zmax, p->dz, p->jerk);
        FDAS_CUDA_TRY(p, cudaGetLastError());
        fdas_twiddle_kernel<double2><<<(p->S + 255) / 256, 256, 0, st>>>((double2 *)p->twiddle, p->S);
    } else {
        if (p->precision == FDAS_F32)
            fdas_bank_kernel<float><<<grid, 256, 0, st>>>(p->bank, p->taps, p->K, p->S, p->T, VC, p->m_max, p->zmax, p->dz, p->jerk);
        else
            fdas_bank_kernel<__nv_bfloat16><<<grid, 256, 0, st>>>(p->bank, p->taps, p->K, p->S, p->T, VC, p->m_max, p->zmax, p->dz, p->jerk);
        FDAS_CUDA_TRY(p, cudaGetLastError());
        fdas_twiddle_kernel<float2><<<(p->S + 255) / 256, 256, 0, st>>>((float2 *)p->twiddle, p->S);
    }
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 3;
    return FDAS_OK;
}
