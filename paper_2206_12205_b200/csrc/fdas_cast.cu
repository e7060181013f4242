// fdas_cast.cu -- the "quick cast" of a bf16-stored power plane (include/fdas.h: fdas_quick_cast).
//
// "the final cast to single-precision ... is completed by copying the two bytes of
// data for each bfloat16 number into the corresponding positions of an all zero single-precision
// output array" -- possible because a bfloat16 is the upper half of an IEEE-754 single
// (Fig. 2).  Here the zero fill and the byte placement are one pass: every output
// word is written once as (bits << 16).  HBM-bound: 2 B read + 4 B written per plane point,
// 128-bit loads (8 bf16) and two 128-bit streaming stores per thread and step.
#include "fdas_internal.h"

namespace {

__global__ void __launch_bounds__(256) fdas_quick_cast_kernel(const unsigned short *__restrict__ src, unsigned *__restrict__ dst,
                                                              long long n)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool aligned = ((reinterpret_cast<uintptr_t>(src) | reinterpret_cast<uintptr_t>(dst)) & 15u) == 0;
    const long long nv = aligned ? n / 8 : 0;
    const uint4 *sv = reinterpret_cast<const uint4 *>(src);
    uint4 *dv = reinterpret_cast<uint4 *>(dst);
    for (long long q = tid; q < nv; q += stride) {
        const uint4 a = __ldcs(sv + q);   // 8 bf16: element 2i in the low half of word i
        __stcs(dv + 2 * q, make_uint4(a.x << 16, a.x & 0xFFFF0000u, a.y << 16, a.y & 0xFFFF0000u));
        __stcs(dv + 2 * q + 1, make_uint4(a.z << 16, a.z & 0xFFFF0000u, a.w << 16, a.w & 0xFFFF0000u));
    }
    for (long long i = nv * 8 + tid; i < n; i += stride) dst[i] = (unsigned)src[i] << 16;
}

}  // namespace

int fdas_launch_quick_cast(fdas_plan *p, const void *src_bf16, void *dst_f32, long long n, cudaStream_t st)
{
    long long want = (n / 8 + 255) / 256;
    const long long cap = (long long)p->num_sms * 8;
    const int grid = (int)(want < cap ? (want > 0 ? want : 1) : cap);
    fdas_quick_cast_kernel<<<grid, 256, 0, st>>>((const unsigned short *)src_bf16, (unsigned *)dst_f32, n);
    FDAS_CUDA_TRY(p, cudaGetLastError());
    p->launches += 1;
    return FDAS_OK;
}
