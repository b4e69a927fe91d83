// Measurement support for bench.py (libsfft_bench.so; never linked into libsfft_b200.so).
// FP64 throughput probes: the peak of the plain
// FP64 FMA pipe (DFMA) and of the FP64 tensor-core path (mma.sync.m8n8k4.f64 -> DMMA) on this device,
// the denominators of the "alu" rooflines in DESIGN.md.  Register-resident operands, 8 independent
// accumulator chains per thread / warp, no memory traffic.
#include <algorithm>

#include "../sfft_internal.h"
#include "sfft_bench.h"

namespace sfft {
namespace {

__global__ void __launch_bounds__(256) k_peak_dfma(double *out, int iters, double a, double b) {
    double c[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) c[q] = threadIdx.x * 1e-9 + q;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int q = 0; q < 8; ++q) c[q] = fma(c[q], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += c[q];
    if (s == 123.456) out[0] = s;
}

__global__ void __launch_bounds__(256) k_peak_dmma(double *out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int q = 0; q < 8; ++q) c[q][0] = c[q][1] = threadIdx.x * 1e-9 + q;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int q = 0; q < 8; ++q)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[q][0]), "+d"(c[q][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += c[q][0] + c[q][1];
    if (s == 123.456) out[0] = s;
}

}  // namespace
}  // namespace sfft

extern "C" int sfft_bench_fp64_peak(int kind, double *tflops) {
    if (!tflops || (kind != 0 && kind != 1)) return SFFT_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return SFFT_ERR_CUDA;
    }
    double *d = nullptr;
    if (cudaMalloc((void **)&d, 8) != cudaSuccess) { cudaGetLastError(); return SFFT_ERR_CUDA; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 20000, blocks = sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) sfft::k_peak_dfma<<<blocks, 256>>>(d, iters, 1.0000001, 1e-9);
        else sfft::k_peak_dmma<<<blocks, 256>>>(d, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        // DFMA: 2 flop per thread-op; DMMA m8n8k4: 2*8*8*4 = 512 flop per warp-op
        const double flop = kind == 0 ? 2.0 * 8 * iters * 256.0 * blocks : 512.0 * 8 * iters * 8.0 * blocks;
        if (rep > 0) best = best > flop / (ms * 1e-3) / 1e12 ? best : flop / (ms * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaError_t e = cudaGetLastError();
    cudaFree(d);
    *tflops = best;
    return e == cudaSuccess ? SFFT_OK : SFFT_ERR_CUDA;
}

extern "C" int sfft_bench_corr_flops(const sfft_plan *p, double *executed, double *tensor) {
    if (!p || !executed || !tensor) return SFFT_ERR_INVALID_ARG;
    if (p->corr_os) {
        // sectioned kernel: per CTA (column slot, x-range part) steps of 4 hops, each 2 FFT64 per sequence and hop
        // (5 N log2 N = 1920 flop) and 4 DMMA (512 flop) per frequency bin
        const int HOP = p->os_hop, hops = (p->H + HOP - 1) / HOP, hpp = (hops + p->Sx - 1) / p->Sx;
        double steps = 0.0;
        for (int xs = 0; xs < p->Sx; ++xs) {
            const int xb = std::min(p->H, xs * hpp * HOP), xe = std::min(p->H, xb + hpp * HOP);
            steps += (xe - xb + 4 * HOP - 1) / (4 * HOP);
        }
        const double ctas = (double)(p->Nh + 1);
        *tensor = ctas * steps * 64.0 * 4.0 * 512.0;
        *executed = *tensor + ctas * steps * (p->nseq * 4.0 * 2.0 * 1920.0) + ctas * p->Sx * 64.0 * 1920.0;
        return SFFT_OK;
    }
    double f = 0.0;
    for (const sfft::CorrJob &j : p->jobs) {
        int rows = 0;
        for (int r = 0; r < j.nrange; ++r) rows += j.xend[r] - j.xbeg[r];
        f += 2.0 * (j.nblk[0] + j.nblk[1]) * 2.0 * 512.0 * (rows / 4) * p->Nh;    // 2 row blocks x blocks x (Re, Im) per 4 rows per column
    }
    *executed = f; *tensor = f;
    return SFFT_OK;
}
