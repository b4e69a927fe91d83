// NEXT-4, FP32 storage / FP64 arithmetic: image widening (float -> double, exact) and narrowing (double -> float,
// round to nearest even) for the host-buffer entry points sfft_run_host*_f32.  HBM-bound streaming kernels,
// 16-byte accesses on the wide side.
#include "sfft_internal.h"

namespace sfft {
namespace {

__global__ void __launch_bounds__(256) k_widen(const float *__restrict__ src, double *__restrict__ dst, size_t count) {
    const size_t i = ((size_t)blockIdx.x * 256 + threadIdx.x) * 4;
    if (i + 3 < count) {
        const float4 v = *reinterpret_cast<const float4 *>(src + i);
        reinterpret_cast<double2 *>(dst + i)[0] = make_double2((double)v.x, (double)v.y);
        reinterpret_cast<double2 *>(dst + i)[1] = make_double2((double)v.z, (double)v.w);
    } else {
        for (size_t k = i; k < count; ++k) dst[k] = (double)src[k];
    }
}

__global__ void __launch_bounds__(256) k_narrow(const double *__restrict__ src, float *__restrict__ dst, size_t count) {
    const size_t i = ((size_t)blockIdx.x * 256 + threadIdx.x) * 4;
    if (i + 3 < count) {
        const double2 a = reinterpret_cast<const double2 *>(src + i)[0], b = reinterpret_cast<const double2 *>(src + i)[1];
        *reinterpret_cast<float4 *>(dst + i) = make_float4((float)a.x, (float)a.y, (float)b.x, (float)b.y);
    } else {
        for (size_t k = i; k < count; ++k) dst[k] = (float)src[k];
    }
}

}  // namespace

cudaError_t launch_widen(sfft_plan *p, const float *src, double *dst, size_t count) {
    k_widen<<<(unsigned)((count + 1023) / 1024), 256, 0, p->stream>>>(src, dst, count);
    p->launches++;
    return cudaGetLastError();
}

cudaError_t launch_narrow(sfft_plan *p, const double *src, float *dst, size_t count) {
    k_narrow<<<(unsigned)((count + 1023) / 1024), 256, 0, p->stream>>>(src, dst, count);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
