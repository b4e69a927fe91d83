// Step a1+a2 (row half): fused y-weighting + real-to-complex FFT along the fast axis.
//
// For every image row x the kernel forms the nKa y-weighted rows g_j(y) R(x,y) (the y-factor
// of the weight T_t = f_i(x) g_j(y); the x-factor f_i(x) is constant along the
// row and is applied later, in the x-direction correlation) plus the row of S, and writes
// their length-W DFTs  r(x,m) = sum_y a(y) exp(-2 pi i m y / W),  m = 0..W/2.
// Layout of the spectrum stack: rhat[b][img][x][m], m in [0, W/2) complex double, with the
// (real) DC and Nyquist bins packed into slot m = 0 as (X[0], X[W/2]).
//
// A real row of length W is transformed as a complex FFT of length W/2 (Stockham autosort,
// radix-4 passes plus one radix-2 pass when log2 is odd, ping-pong in shared memory)
// followed by the even/odd split.  HBM-bound: one 16-byte load and one 16-byte store per
// complex point, both fully coalesced.
#include "fft_regs.cuh"
#include "sfft_internal.h"

namespace sfft {
namespace {

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// One Stockham pass of radix R over N points held in shared memory (forward transform).
// tw[k] = exp(-2 pi i k / (2N)) (the plan's W-point table, W = 2N), so exp(-2 pi i q / N) = tw[2q].
template <int N, int T, int R>
__device__ __forceinline__ void stockham_pass(const double2 *__restrict__ in, double2 *__restrict__ out, int Ns,
                                              const double2 *__restrict__ tw) {
    for (int j = threadIdx.x; j < N / R; j += T) {
        const int k = j & (Ns - 1);
        double2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = in[j + r * (N / R)];
        if (Ns > 1) {
            const int step = 2 * (N / (Ns * R)) * k;   // index of exp(-2 pi i k /(Ns R)) in the W-point table
#pragma unroll
            for (int r = 1; r < R; ++r) v[r] = cmul(v[r], __ldg(&tw[r * step]));
        }
        const int j0 = (j - k) * R + k;
        if (R == 4) {
            double2 t0 = make_double2(v[0].x + v[2].x, v[0].y + v[2].y);
            double2 t1 = make_double2(v[0].x - v[2].x, v[0].y - v[2].y);
            double2 t2 = make_double2(v[1].x + v[3].x, v[1].y + v[3].y);
            double2 d = make_double2(v[1].x - v[3].x, v[1].y - v[3].y);
            double2 t3 = make_double2(d.y, -d.x);   // -i * (v1 - v3)
            out[j0] = make_double2(t0.x + t2.x, t0.y + t2.y);
            out[j0 + Ns] = make_double2(t1.x + t3.x, t1.y + t3.y);
            out[j0 + 2 * Ns] = make_double2(t0.x - t2.x, t0.y - t2.y);
            out[j0 + 3 * Ns] = make_double2(t1.x - t3.x, t1.y - t3.y);
        } else {
            out[j0] = make_double2(v[0].x + v[1].x, v[0].y + v[1].y);
            out[j0 + Ns] = make_double2(v[0].x - v[1].x, v[0].y - v[1].y);
        }
    }
}

template <int N>
struct Log2 { static constexpr int value = 1 + Log2<N / 2>::value; };
template <>
struct Log2<1> { static constexpr int value = 0; };

// Forward complex FFT of N points in shared memory; returns the buffer holding the result.
template <int N, int T>
__device__ __forceinline__ double2 *fft_smem_forward(double2 *a, double2 *b, const double2 *__restrict__ tw) {
    constexpr int LOG = Log2<N>::value;
    int Ns = 1;
    double2 *in = a, *out = b;
#pragma unroll
    for (int s = 0; s < LOG / 2; ++s) {
        stockham_pass<N, T, 4>(in, out, Ns, tw);
        __syncthreads();
        Ns *= 4;
        double2 *t = in; in = out; out = t;
    }
    if (LOG & 1) {
        stockham_pass<N, T, 2>(in, out, Ns, tw);
        __syncthreads();
        double2 *t = in; in = out; out = t;
    }
    return in;
}

// grid: x = image slot (0..nKa-1: weighted R rows, nKa: S), y = row, z = batch entry
template <int NH, int T>
__global__ void __launch_bounds__(T) k_rowfft_forward(const double *__restrict__ R, const double *__restrict__ S,
                                                      const double *__restrict__ gK, const double2 *__restrict__ twW,
                                                      double2 *__restrict__ rhat, int H, int nKa) {
    extern __shared__ double2 sm[];
    double2 *a = sm, *b = sm + NH;
    constexpr int W = 2 * NH;
    const int img = blockIdx.x, x = blockIdx.y, bz = blockIdx.z;
    const double2 *src = reinterpret_cast<const double2 *>((img < nKa ? R : S) + ((size_t)bz * H + x) * W);
    if (img < nKa) {
        const double2 *g = reinterpret_cast<const double2 *>(gK + (size_t)img * W);
        for (int i = threadIdx.x; i < NH; i += T) {
            double2 v = __ldg(&src[i]), gg = __ldg(&g[i]);
            a[i] = make_double2(v.x * gg.x, v.y * gg.y);    // z[n] = a[2n] + i a[2n+1]
        }
    } else {
        for (int i = threadIdx.x; i < NH; i += T) a[i] = __ldg(&src[i]);
    }
    __syncthreads();
    const double2 *Z = fft_smem_forward<NH, T>(a, b, twW);
    double2 *dst = rhat + (((size_t)bz * (nKa + 1) + img) * H + x) * NH;
    // even/odd split: E = (Z[k] + conj Z[NH-k])/2, O = (Z[k] - conj Z[NH-k])/(2i), X[k] = E + w^k O,
    // X[NH-k] = conj(E - w^k O), w = exp(-2 pi i / W)
    for (int k = threadIdx.x; k <= NH / 2; k += T) {
        if (k == 0) {
            double2 z0 = Z[0];
            dst[0] = make_double2(z0.x + z0.y, z0.x - z0.y);   // (X[0], X[W/2]) packed
        } else {
            double2 zk = Z[k], zn = Z[NH - k];
            double2 E = make_double2(0.5 * (zk.x + zn.x), 0.5 * (zk.y - zn.y));
            double2 O = make_double2(0.5 * (zk.y + zn.y), -0.5 * (zk.x - zn.x));
            double2 wO = cmul(__ldg(&twW[k]), O);
            dst[k] = make_double2(E.x + wO.x, E.y + wO.y);
            if (k != NH - k) dst[NH - k] = make_double2(E.x - wO.x, -(E.y - wO.y));
        }
    }
}

template <int NH>
cudaError_t launch_fwd(sfft_plan *p, const double *dR, const double *dS) {
    constexpr int T = NH >= 1024 ? 256 : (NH >= 256 ? 128 : 64);
    size_t smem = 2 * (size_t)NH * sizeof(double2);
    auto kern = k_rowfft_forward<NH, T>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(dS ? p->nimg : p->nKa, p->H, p->nbatch);     // dS == nullptr: the weighted R rows only
    kern<<<grid, T, smem, p->stream>>>(dR, dS, p->dt.gK, p->dt.twW, p->rhat, p->H, p->nKa);
    p->launches++;
    return cudaGetLastError();
}

// Register-tiled variant for NH >= 512 (fft_regs.cuh): three radix-16/16/R3 passes, RPC rows per CTA.
// grid: x = image slot, y = row group, z = batch entry; block: (NH/16, RPC).
template <int NH>
__global__ void __launch_bounds__(FftCfg<NH>::T * (FftCfg<NH>::T >= 128 ? 1 : 128 / FftCfg<NH>::T))
k_rowfft_forward16(const double *__restrict__ R, const double *__restrict__ S, const double *__restrict__ gK,
                   const double2 *__restrict__ twW, double2 *__restrict__ rhat, int H, int nKa, int poly) {
    using C = FftCfg<NH>;
    constexpr int T = C::T, RPC = T >= 128 ? 1 : 128 / T, W = 2 * NH;
    extern __shared__ double2 sm2[];
    double2 *tw2 = sm2, *buf = sm2 + C::TW2 + threadIdx.y * C::BUF;
    const int tid = threadIdx.x, img = blockIdx.x, x = blockIdx.y * RPC + threadIdx.y, bz = blockIdx.z;
    if (threadIdx.y == 0) fft_load_tw2<NH>(tw2, twW);
    // (H need not be a multiple of RPC: a row slot past the end transforms the last row again and stores nothing)
    const double2 *src = reinterpret_cast<const double2 *>((img < nKa ? R : S) + ((size_t)bz * H + min(x, H - 1)) * W);
    double2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) v[r] = __ldg(&src[tid + r * T]);          // z[n] = a[2n] + i a[2n+1]
    if (img < nKa && poly) {
        // g_j(y) = u_y^j with u_y = (2y+1)/W - 1 exact in double: no table traffic (the kernel is bound by the
        // L1/shared data pipe); j = 0 needs no multiplication at all
        if (img > 0) {
            constexpr double invW = 1.0 / W;
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int nn = tid + r * T;
                const double u0 = (double)(4 * nn + 1) * invW - 1.0, u1 = (double)(4 * nn + 3) * invW - 1.0;
                double w0 = u0, w1 = u1;
                for (int j = 1; j < img; ++j) { w0 *= u0; w1 *= u1; }
                v[r].x *= w0;
                v[r].y *= w1;
            }
        }
    } else if (img < nKa) {
        const double2 *g = reinterpret_cast<const double2 *>(gK + (size_t)img * W);
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const double2 gg = __ldg(&g[tid + r * T]);
            v[r].x *= gg.x;
            v[r].y *= gg.y;
        }
    }
    __syncthreads();                                                       // tw2 visible
    fft_core<NH, false>(v, buf, tw2, twW);
    // Even/odd split (see k_rowfft_forward) from the registers of the last pass: this thread holds Z[k + 256 r] of its
    // butterflies k = tid + T q, whose partners Z[NH - k - 256 r] belong to butterfly 256 - k (k = 0: to itself, at
    // R3 - r; k = 128: to itself, at R3 - 1 - r).  Only the butterflies k >= 128 (and k = 0) go through shared memory,
    // those with k <= 128 read their partners and produce both X[idx] and X[NH - idx]: half the exchange of a full
    // write and read of the spectrum.  Slot of (k, r): buf[r * 257 + k] (conflict-free in k).
    constexpr int R3 = C::R3, NB3 = C::NB3;
#pragma unroll
    for (int q = 0; q < NB3; ++q) {
        const int k = tid + T * q;
        if (k >= 128 || k == 0) {
#pragma unroll
            for (int r = 0; r < R3; ++r) buf[r * 257 + k] = v[q * R3 + r];
        }
    }
    __syncthreads();
    double2 *dst = rhat + (((size_t)bz * (nKa + 1) + img) * H + x) * NH;
    if (x < H) {
#pragma unroll
        for (int q = 0; q < NB3; ++q) {
            const int k = tid + T * q;
            if (k > 128) continue;
#pragma unroll
            for (int r = 0; r < R3; ++r) {
                const int idx = k + 256 * r;
                const double2 zk = v[q * R3 + r];
                if (idx == 0) {
                    dst[0] = make_double2(zk.x + zk.y, zk.x - zk.y);
                    continue;
                }
                // partner Z[NH - idx]
                const double2 zn = k == 0 ? buf[(R3 - r) * 257] : (k == 128 ? buf[(R3 - 1 - r) * 257 + 128] : buf[(R3 - 1 - r) * 257 + 256 - k]);
                const double2 E = make_double2(0.5 * (zk.x + zn.x), 0.5 * (zk.y - zn.y));
                const double2 O = make_double2(0.5 * (zk.y + zn.y), -0.5 * (zk.x - zn.x));
                const double2 wO = cmul(__ldg(&twW[idx]), O);
                dst[idx] = make_double2(E.x + wO.x, E.y + wO.y);
                if (idx != NH - idx) dst[NH - idx] = make_double2(E.x - wO.x, -(E.y - wO.y));
            }
        }
    }
}

template <int NH>
cudaError_t launch_fwd16(sfft_plan *p, const double *dR, const double *dS) {
    using C = FftCfg<NH>;
    constexpr int T = C::T, RPC = T >= 128 ? 1 : 128 / T;
    const size_t smem = (size_t)(C::TW2 + RPC * C::BUF) * sizeof(double2);
    auto kern = k_rowfft_forward16<NH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(dS ? p->nimg : p->nKa, (p->H + RPC - 1) / RPC, p->nbatch);
    kern<<<grid, dim3(T, RPC), smem, p->stream>>>(dR, dS, p->dt.gK, p->dt.twW, p->rhat, p->H, p->nKa,
                                                  p->basis == SFFT_BASIS_POLY);
    p->launches++;
    return cudaGetLastError();
}

// W not a power of two (W even; true survey frames, e.g. 2046 x 4094): the complex N = W/2 point DFT of
// z[n] = a[2n] + i a[2n+1] is run as a chirp-z (Bluestein) transform on the register FFT of fft_regs.cuh,
//   Z[k] = c[k] sum_n (z[n] c[n]) conj(c[k-n]),  c[n] = exp(-i pi n^2 / N),
// i.e. a circular convolution of length M = 2^k >= 2N - 1:  conv = IFFT_M( FFT_M(z c) * bhat ),  bhat = FFT_M(conj c
// wrapped) a plan table, with the inverse transform taken as conj(FFT_M(conj .)) / M.  The even/odd split that follows
// is the one of the power-of-two kernels with N in place of NH.  One CTA of M/16 threads per image row and image.
// grid: x = image slot, y = row, z = batch entry.
template <int M>
__global__ void __launch_bounds__(FftCfg<M>::T)
k_rowfft_forward_bs(const double *__restrict__ R, const double *__restrict__ S, const double *__restrict__ gK,
                    const double2 *__restrict__ twW, const double2 *__restrict__ twM, const double2 *__restrict__ chirp,
                    const double2 *__restrict__ bhat, double2 *__restrict__ rhat, int H, int W, int nKa) {
    using C = FftCfg<M>;
    constexpr int T = C::T;
    extern __shared__ double2 sm3[];
    double2 *tw2 = sm3, *buf = sm3 + C::TW2, *zs = buf + C::BUF;     // zs[N]: the N-point spectrum for the split
    const int tid = threadIdx.x, img = blockIdx.x, x = blockIdx.y, bz = blockIdx.z, N = W / 2;
    fft_load_tw2<M>(tw2, twM);
    const double2 *src = reinterpret_cast<const double2 *>((img < nKa ? R : S) + ((size_t)bz * H + x) * W);
    const double2 *g = reinterpret_cast<const double2 *>(gK + (size_t)(img < nKa ? img : 0) * W);
    double2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int n = tid + r * T;
        v[r] = make_double2(0.0, 0.0);
        if (n < N) {
            double2 a = __ldg(&src[n]);
            if (img < nKa) { const double2 gg = __ldg(&g[n]); a.x *= gg.x; a.y *= gg.y; }
            v[r] = cmul(a, __ldg(&chirp[n]));
        }
    }
    __syncthreads();                                                       // tw2 visible
    fft_core<M>(v, buf, tw2, twM);
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int n = tid + r * T;
        const double2 t = cmul(buf[n], __ldg(&bhat[n]));
        v[r] = make_double2(t.x, -t.y);
    }
    __syncthreads();                                                       // buf consumed before it is rewritten
    fft_core<M>(v, buf, tw2, twM);
    constexpr double invM = 1.0 / M;
    for (int k = tid; k < N; k += T) {
        const double2 u = buf[k], c = __ldg(&chirp[k]);
        zs[k] = cmul(make_double2(u.x * invM, -u.y * invM), c);
    }
    __syncthreads();
    double2 *dst = rhat + (((size_t)bz * (nKa + 1) + img) * H + x) * N;
    // even/odd split (see k_rowfft_forward), w = exp(-2 pi i / W)
    for (int k = tid; k <= N / 2; k += T) {
        if (k == 0) {
            const double2 z0 = zs[0];
            dst[0] = make_double2(z0.x + z0.y, z0.x - z0.y);
        } else {
            const double2 zk = zs[k], zn = zs[N - k];
            const double2 E = make_double2(0.5 * (zk.x + zn.x), 0.5 * (zk.y - zn.y));
            const double2 O = make_double2(0.5 * (zk.y + zn.y), -0.5 * (zk.x - zn.x));
            const double2 wO = cmul(__ldg(&twW[k]), O);
            dst[k] = make_double2(E.x + wO.x, E.y + wO.y);
            if (k != N - k) dst[N - k] = make_double2(E.x - wO.x, -(E.y - wO.y));
        }
    }
}

template <int M>
cudaError_t launch_fwd_bs(sfft_plan *p, const double *dR, const double *dS) {
    using C = FftCfg<M>;
    const size_t smem = (size_t)(C::TW2 + C::BUF + p->Nh) * sizeof(double2);
    auto kern = k_rowfft_forward_bs<M>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(dS ? p->nimg : p->nKa, p->H, p->nbatch);
    kern<<<grid, C::T, smem, p->stream>>>(dR, dS, p->dt.gK, p->dt.twW, p->dt.twM, p->dt.chirp, p->dt.bhat, p->rhat, p->H, p->W,
                                          p->nKa);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_rowfft_forward(sfft_plan *p, const double *dR, const double *dS) {
    switch (p->bsM) {
        case 0: break;
        case 512: return launch_fwd_bs<512>(p, dR, dS);
        case 1024: return launch_fwd_bs<1024>(p, dR, dS);
        case 2048: return launch_fwd_bs<2048>(p, dR, dS);
        case 4096: return launch_fwd_bs<4096>(p, dR, dS);
        default: return cudaErrorInvalidValue;
    }
    switch (p->Nh) {
        case 32: return launch_fwd<32>(p, dR, dS);
        case 64: return launch_fwd<64>(p, dR, dS);
        case 128: return launch_fwd<128>(p, dR, dS);
        case 256: return launch_fwd<256>(p, dR, dS);
        case 512: return launch_fwd16<512>(p, dR, dS);
        case 1024: return launch_fwd16<1024>(p, dR, dS);
        case 2048: return launch_fwd16<2048>(p, dR, dS);
        case 4096: return launch_fwd16<4096>(p, dR, dS);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace sfft
