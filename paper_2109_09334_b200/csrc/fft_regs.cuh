// Register-resident FFT building blocks shared by the row-transform kernels (rowfft.cu, subtract_fourier.cu).
//
// A complex FFT of NH = 256 * R3 points (R3 = 2, 4, 8, 16; NH = 512 .. 4096) is run by NH/16 threads holding
// 16 points each, as three Stockham autosort passes of radix 16, 16, R3.  The butterflies of a pass live
// entirely in registers (fft_reg<R>), so a transform costs three shared-memory exchanges instead of
// log2(NH)/2 radix-4 passes through shared memory.  Pass 1 writes 16 consecutive points per thread; that
// buffer is padded by one element per 16 (index i -> i + i/16) to keep the 128-bit stores conflict-free.
#pragma once
#include <cuda_runtime.h>

namespace sfft {

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmulf(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ double2 mul_mi(double2 a) { return make_double2(a.y, -a.x); }   // a * (-i)

// Forward DFT (kernel exp(-2 pi i jk/R)) of R points in registers, natural order in and out.
template <int R>
__device__ __forceinline__ void fft_reg(double2 (&v)[R]);

template <>
__device__ __forceinline__ void fft_reg<2>(double2 (&v)[2]) {
    const double2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
}

template <>
__device__ __forceinline__ void fft_reg<4>(double2 (&v)[4]) {
    const double2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]), t2 = cadd(v[1], v[3]), t3 = mul_mi(csub(v[1], v[3]));
    v[0] = cadd(t0, t2);
    v[1] = cadd(t1, t3);
    v[2] = csub(t0, t2);
    v[3] = csub(t1, t3);
}

template <>
__device__ __forceinline__ void fft_reg<8>(double2 (&v)[8]) {
    constexpr double h = 0.70710678118654752440;
    double2 e[4] = {v[0], v[2], v[4], v[6]}, o[4] = {v[1], v[3], v[5], v[7]};
    fft_reg<4>(e);
    fft_reg<4>(o);
    o[1] = make_double2(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x));      // * (1 - i)/sqrt2
    o[2] = mul_mi(o[2]);
    o[3] = make_double2(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y));     // * (-1 - i)/sqrt2
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        v[k] = cadd(e[k], o[k]);
        v[k + 4] = csub(e[k], o[k]);
    }
}

template <>
__device__ __forceinline__ void fft_reg<16>(double2 (&v)[16]) {
    constexpr double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173, h = 0.70710678118654752440;
    double2 e[8], o[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
    fft_reg<8>(e);
    fft_reg<8>(o);
    // o[k] *= exp(-2 pi i k / 16)
    o[1] = cmulf(o[1], make_double2(c1, -s1));
    o[2] = make_double2(h * (o[2].x + o[2].y), h * (o[2].y - o[2].x));
    o[3] = cmulf(o[3], make_double2(s1, -c1));
    o[4] = mul_mi(o[4]);
    o[5] = cmulf(o[5], make_double2(-s1, -c1));
    o[6] = make_double2(h * (o[6].y - o[6].x), -h * (o[6].x + o[6].y));
    o[7] = cmulf(o[7], make_double2(-c1, -s1));
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = cadd(e[k], o[k]);
        v[k + 8] = csub(e[k], o[k]);
    }
}

template <int NH>
struct FftCfg {
    static_assert(NH == 512 || NH == 1024 || NH == 2048 || NH == 4096, "NH = 256 * {2,4,8,16}");
    static constexpr int T = NH / 16;                    // threads per transform
    static constexpr int R3 = NH / 256;                  // radix of the last pass
    static constexpr int NB3 = 16 / R3;                  // last-pass butterflies per thread
    static constexpr int BUF = NH + NH / 16;             // double2 elements of the exchange buffer
    static constexpr int TW2 = 256;                      // pass-2 twiddle table tw2[r*16 + k] = exp(-2 pi i k r / 256)
    static constexpr size_t SMEM = (size_t)(BUF + TW2) * sizeof(double2);
};

// Fill the pass-2 twiddle table from the plan's W-point table twW[q] = exp(-2 pi i q / W), W = 2 NH.
template <int NH>
__device__ __forceinline__ void fft_load_tw2(double2 *tw2, const double2 *__restrict__ twW) {
    for (int i = threadIdx.x; i < 256; i += FftCfg<NH>::T) {
        const int r = i >> 4, k = i & 15;
        tw2[i] = __ldg(&twW[(k * r) * (2 * NH / 256)]);
    }
}

// Forward FFT of NH points: on entry v[r] = z[tid + r*T]; on exit the spectrum Z[0..NH) is in buf (natural
// order, unpadded) and visible to all threads.  buf must not be in use by other threads on entry (the
// caller separates calls by a barrier).
// STORE = false: the last pass leaves its results in registers instead, v[q*R3 + r] = Z[k + 256 r] with
// k = tid + T q (q < NB3, r < R3), and buf is free again on exit.
template <int NH, bool STORE = true>
__device__ __forceinline__ void fft_core(double2 (&v)[16], double2 *buf, const double2 *tw2,
                                         const double2 *__restrict__ twW) {
    using C = FftCfg<NH>;
    constexpr int T = C::T, R3 = C::R3, NB3 = C::NB3;
    const int tid = threadIdx.x;
    // pass 1: radix 16, Ns = 1
    fft_reg<16>(v);
#pragma unroll
    for (int r = 0; r < 16; ++r) buf[17 * tid + r] = v[r];          // index 16 tid + r, padded
    __syncthreads();
    // pass 2: radix 16, Ns = 16
    const int k2 = tid & 15;
#pragma unroll
    for (int r = 0; r < 16; ++r) { const int i = tid + r * T; v[r] = buf[i + (i >> 4)]; }
    {
        // twiddles exp(-2 pi i k2 r / 256) = w^r from ONE table read by a shallow product tree (depth 4): the kernels
        // using this are bound by the shared-memory data pipe, not by FP64 issue, so 14 complex products are
        // cheaper than 14 more 16-byte shared loads per thread
        const double2 w1 = tw2[16 + k2], w2 = cmulf(w1, w1), w3 = cmulf(w2, w1), w4 = cmulf(w2, w2);
        const double2 w5 = cmulf(w4, w1), w6 = cmulf(w4, w2), w7 = cmulf(w4, w3), w8 = cmulf(w4, w4);
        v[1] = cmulf(v[1], w1); v[2] = cmulf(v[2], w2); v[3] = cmulf(v[3], w3); v[4] = cmulf(v[4], w4);
        v[5] = cmulf(v[5], w5); v[6] = cmulf(v[6], w6); v[7] = cmulf(v[7], w7); v[8] = cmulf(v[8], w8);
        v[9] = cmulf(v[9], cmulf(w8, w1)); v[10] = cmulf(v[10], cmulf(w8, w2)); v[11] = cmulf(v[11], cmulf(w8, w3));
        v[12] = cmulf(v[12], cmulf(w8, w4)); v[13] = cmulf(v[13], cmulf(w8, w5)); v[14] = cmulf(v[14], cmulf(w8, w6));
        v[15] = cmulf(v[15], cmulf(w8, w7));
    }
    fft_reg<16>(v);
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 16; ++r) buf[(tid - k2) * 16 + k2 + 16 * r] = v[r];
    __syncthreads();
    // pass 3: radix R3, Ns = 256; NB3 butterflies per thread
#pragma unroll
    for (int q = 0; q < NB3; ++q)
#pragma unroll
        for (int r = 0; r < R3; ++r) v[q * R3 + r] = buf[tid + T * q + r * (NH / R3)];
    __syncthreads();
#pragma unroll
    for (int q = 0; q < NB3; ++q) {
        const int j = tid + T * q, k = j & 255;
        double2 u[R3];
#pragma unroll
        for (int r = 0; r < R3; ++r) u[r] = v[q * R3 + r];
        // twiddles exp(-2 pi i k r / NH) = w^r from w = twW[2k] by a shallow product tree
        const double2 w1 = __ldg(&twW[2 * k]);
        u[1] = cmulf(u[1], w1);
        if constexpr (R3 >= 4) {
            const double2 w2 = cmulf(w1, w1), w3 = cmulf(w2, w1);
            u[2] = cmulf(u[2], w2);
            u[3] = cmulf(u[3], w3);
            if constexpr (R3 >= 8) {
                const double2 w4 = cmulf(w2, w2), w5 = cmulf(w4, w1), w6 = cmulf(w4, w2), w7 = cmulf(w4, w3);
                u[4] = cmulf(u[4], w4);
                u[5] = cmulf(u[5], w5);
                u[6] = cmulf(u[6], w6);
                u[7] = cmulf(u[7], w7);
                if constexpr (R3 >= 16) {
                    const double2 w8 = cmulf(w4, w4);
                    u[8] = cmulf(u[8], w8);
                    u[9] = cmulf(u[9], cmulf(w8, w1));
                    u[10] = cmulf(u[10], cmulf(w8, w2));
                    u[11] = cmulf(u[11], cmulf(w8, w3));
                    u[12] = cmulf(u[12], cmulf(w8, w4));
                    u[13] = cmulf(u[13], cmulf(w8, w5));
                    u[14] = cmulf(u[14], cmulf(w8, w6));
                    u[15] = cmulf(u[15], cmulf(w8, w7));
                }
            }
        }
        fft_reg<R3>(u);
#pragma unroll
        for (int r = 0; r < R3; ++r) {
            if (STORE) buf[(j - k) * R3 + k + 256 * r] = u[r];      // (T NB3 = 256: j = k, the index is k + 256 r)
            else v[q * R3 + r] = u[r];
        }
    }
    if (STORE) __syncthreads();
}

}  // namespace sfft
