// fdas_fft.cuh -- in-register radix-2/4/8/16 DFT butterflies (inverse sign, exp(+2 pi i ..))
// used by the fused convolve kernel.  A forward transform is obtained from the same code by
// swapping real and imaginary parts on the way in and out: FFT(x) = swap(IFFT(swap(x))).
//
// Every function works on fully unrolled register arrays re[], im[]; the result X[k] of an
// R-point transform is left in slot DftSlot<R>::of(k) (no data movement for the digit
// reversal: the caller indexes through of()).
#pragma once
#include <cuda_runtime.h>

namespace fdas {

template <typename T> struct Cst;
template <> struct Cst<float> {
    static constexpr float R = 0.70710678118654752440f;   // cos(pi/4)
    static constexpr float C1 = 0.92387953251128675613f;  // cos(pi/8)
    static constexpr float S1 = 0.38268343236508977173f;  // sin(pi/8)
};
template <> struct Cst<double> {
    static constexpr double R = 0.70710678118654752440;
    static constexpr double C1 = 0.92387953251128675613;
    static constexpr double S1 = 0.38268343236508977173;
};

// (xr + i xi) *= (wr + i wi)
template <typename T>
__device__ __forceinline__ void cmul(T &xr, T &xi, T wr, T wi)
{
    T tr = xr * wr - xi * wi;
    T ti = xr * wi + xi * wr;
    xr = tr;
    xi = ti;
}

// 4-point inverse-sign DFT in place: X0->s0, X1->s1, X2->s2, X3->s3  (w4 = +i)
template <typename T>
__device__ __forceinline__ void dft4(T &r0, T &i0, T &r1, T &i1, T &r2, T &i2, T &r3, T &i3)
{
    T ar = r0 + r2, ai = i0 + i2;
    T br = r0 - r2, bi = i0 - i2;
    T cr = r1 + r3, ci = i1 + i3;
    T dr = r1 - r3, di = i1 - i3;
    r0 = ar + cr; i0 = ai + ci;
    r2 = ar - cr; i2 = ai - ci;
    r1 = br - di; i1 = bi + dr;   // b + i d
    r3 = br + di; i3 = bi - dr;   // b - i d
}

template <typename T>
__device__ __forceinline__ void dft2(T &r0, T &i0, T &r1, T &i1)
{
    T ar = r0 + r1, ai = i0 + i1;
    r1 = r0 - r1; i1 = i0 - i1;
    r0 = ar; i0 = ai;
}

template <int R> struct DftSlot;
template <> struct DftSlot<1> { __host__ __device__ static constexpr int of(int k) { return k; } };
template <> struct DftSlot<2> { __host__ __device__ static constexpr int of(int k) { return k; } };
template <> struct DftSlot<4> { __host__ __device__ static constexpr int of(int k) { return k; } };
template <> struct DftSlot<8> { __host__ __device__ static constexpr int of(int k) { return 2 * (k & 3) + (k >> 2); } };
template <> struct DftSlot<16> { __host__ __device__ static constexpr int of(int k) { return 4 * (k & 3) + (k >> 2); } };

template <typename T, int R> struct Dft;

template <typename T> struct Dft<T, 1> {
    __device__ __forceinline__ static void run(T *, T *) {}
};
template <typename T> struct Dft<T, 2> {
    __device__ __forceinline__ static void run(T *re, T *im) { dft2(re[0], im[0], re[1], im[1]); }
};
template <typename T> struct Dft<T, 4> {
    __device__ __forceinline__ static void run(T *re, T *im)
    {
        dft4(re[0], im[0], re[1], im[1], re[2], im[2], re[3], im[3]);
    }
};

// 8 = 4 x 2:  a = 2 a1 + a2,  k = k1 + 4 k2
template <typename T> struct Dft<T, 8> {
    __device__ __forceinline__ static void run(T *re, T *im)
    {
        constexpr T R = Cst<T>::R;
        dft4(re[0], im[0], re[2], im[2], re[4], im[4], re[6], im[6]);
        dft4(re[1], im[1], re[3], im[3], re[5], im[5], re[7], im[7]);
        // slot 2 k1 + 1 *= w8^k1
        {   // k1 = 1: (R, R)
            T tr = (re[3] - im[3]) * R, ti = (re[3] + im[3]) * R;
            re[3] = tr; im[3] = ti;
        }
        {   // k1 = 2: +i
            T tr = -im[5], ti = re[5];
            re[5] = tr; im[5] = ti;
        }
        {   // k1 = 3: (-R, R)
            T tr = -(re[7] + im[7]) * R, ti = (re[7] - im[7]) * R;
            re[7] = tr; im[7] = ti;
        }
        dft2(re[0], im[0], re[1], im[1]);
        dft2(re[2], im[2], re[3], im[3]);
        dft2(re[4], im[4], re[5], im[5]);
        dft2(re[6], im[6], re[7], im[7]);
    }
};

// 16 = 4 x 4:  a = 4 a1 + a2,  k = k1 + 4 k2
template <typename T> struct Dft<T, 16> {
    __device__ __forceinline__ static void run(T *re, T *im)
    {
        constexpr T R = Cst<T>::R, C1 = Cst<T>::C1, S1 = Cst<T>::S1;
#pragma unroll
        for (int a2 = 0; a2 < 4; ++a2)
            dft4(re[a2], im[a2], re[4 + a2], im[4 + a2], re[8 + a2], im[8 + a2], re[12 + a2], im[12 + a2]);
        // slot 4 k1 + a2 *= w16^(a2 k1)
        cmul(re[5], im[5], C1, S1);                       // e = 1
        {   // e = 2: (R, R)
            T tr = (re[6] - im[6]) * R, ti = (re[6] + im[6]) * R;
            re[6] = tr; im[6] = ti;
        }
        cmul(re[7], im[7], S1, C1);                       // e = 3
        {   // slot 9 (k1=2,a2=1): e = 2
            T tr = (re[9] - im[9]) * R, ti = (re[9] + im[9]) * R;
            re[9] = tr; im[9] = ti;
        }
        {   // slot 10: e = 4: +i
            T tr = -im[10], ti = re[10];
            re[10] = tr; im[10] = ti;
        }
        {   // slot 11: e = 6: (-R, R)
            T tr = -(re[11] + im[11]) * R, ti = (re[11] - im[11]) * R;
            re[11] = tr; im[11] = ti;
        }
        cmul(re[13], im[13], S1, C1);                     // slot 13 (k1=3,a2=1): e = 3
        {   // slot 14: e = 6
            T tr = -(re[14] + im[14]) * R, ti = (re[14] - im[14]) * R;
            re[14] = tr; im[14] = ti;
        }
        cmul(re[15], im[15], -C1, -S1);                   // slot 15: e = 9
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1)
            dft4(re[4 * k1], im[4 * k1], re[4 * k1 + 1], im[4 * k1 + 1], re[4 * k1 + 2], im[4 * k1 + 2],
                 re[4 * k1 + 3], im[4 * k1 + 3]);
    }
};

}  // namespace fdas
