// Steps a7+a8, Fourier route (Eq. 13, 208-212; Eqs. 1, 12): the spatially varying
// convolution evaluated on the row spectra, used when it needs fewer FP64 operations than the direct
// tensor-core contraction of subtract.cu (wide kernels, few spatial terms; see subtract_use_fourier).
//
// With R^t = f_i(x) g_j(y) R and r_j(x,m) the length-W row DFT of g_j R (rowfft.cu), shifting by beta
// along y multiplies a row spectrum by exp(-2 pi i m beta / W), so the row DFT of the model image
//   Mdl(x,y) = sum_t sum_{a,b} k_{t,ab} R^t(x-a, y-b)                       (k: pixel kernel, Eqs. 3-4)
// is a short FIR filter along x, independently for every spectrum column m:
//   mdl(x,m) = sum_a sum_t khat_{t,a}(m) f_i(x-a) r_j(x-a, m),   khat_{t,a}(m) = sum_b k_{t,ab} exp(-2 pi i m b / W).
// That is L*FK complex multiply-adds per spectrum point (102 at config 4) against L*L*nKa real ones
// per pixel for the direct form (867; 1248 executed).  Then one inverse row transform gives the model
// and D = S - Mdl - sum_s b_s T'_s is formed in its epilogue.
//
//   k_kernel_spectrum : khat[b][(a,t)][m] from the folded pixel kernels (17-term DFTs)
//   k_fir_x           : the FIR filter; one thread per column m walks down x with the L+3 partial
//                       outputs of a 4-row step in registers (FP64 FMA pipe bound); the packed
//                       DC/Nyquist column runs the same code as two real filters
//   k_rowfft_inverse_sub : complex-to-real inverse row FFT (conjugate trick on the forward
//                       radix-16 passes of fft_regs.cuh) fused with the difference (HBM bound)
#include "fft_regs.cuh"
#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int kFirCols = 32;     // spectrum columns per CTA of k_fir_x (one warp = one x-range of 32 columns)
constexpr int kFirWarps = 4;     // x-ranges per CTA
constexpr int kFirMaxFK = 48;
constexpr int kFirMaxNKa = 8;    // x-basis functions of the FIR route (their 4-row weight tiles live in shared memory)

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// khat[b][ai*FK + t][m] = sum_bi kfold[b][t][ai][bi] exp(-2 pi i m (bi - w) / W); column 0 packs the two
// real values (m = 0, m = W/2).  grid: x = column block of 128, y = (ai, t), z = batch.
__global__ void k_kernel_spectrum(const double *__restrict__ kfold, const double2 *__restrict__ twW,
                                  double2 *__restrict__ khat, int Nh, int L, int FK) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, ai = blockIdx.y / FK, t = blockIdx.y - ai * FK, b = blockIdx.z;
    if (m >= Nh) return;
    const int w = (L - 1) / 2, W = 2 * Nh, wmask = (W & (W - 1)) == 0 ? W - 1 : -1;
    const double *k = kfold + (((size_t)b * FK + t) * L + ai) * L;
    double re = 0.0, im = 0.0;
    if (m == 0) {
        for (int bi = 0; bi < L; ++bi) {
            const double v = __ldg(&k[bi]);
            re += v;
            im += ((bi - w) & 1) ? -v : v;              // exp(-i pi beta) = (-1)^beta
        }
    } else {
        for (int bi = 0; bi < L; ++bi) {
            const double v = __ldg(&k[bi]);
            const double2 tw = __ldg(&twW[wrap_index(m * (bi - w), W, wmask)]);
            re = fma(v, tw.x, re);
            im = fma(v, tw.y, im);
        }
    }
    khat[((size_t)b * L * FK + blockIdx.y) * Nh + m] = make_double2(re, im);
}

// acc += k z for a complex column; for the packed column 0 (two real filters: DC in .x, Nyquist in .y)
// the caller passes (kb, kc, kd) = (0, k.y, 0) instead of (-k.y, k.x, k.y), giving acc += (k.x z.x, k.y z.y).
__device__ __forceinline__ void cmac(double2 &acc, double ka, double kb, double kc, double kd, const double2 z) {
    acc.x = fma(ka, z.x, acc.x);
    acc.y = fma(kc, z.y, acc.y);
    acc.x = fma(kb, z.y, acc.x);
    acc.y = fma(kd, z.x, acc.y);
}

struct FirDims { int H, Nh, nimg, nKa, FK, NO, pad; };

// grid: x = block of 32 columns, y = group of 4 x-ranges, z = batch.  block: 128 (warp = x-range).
// Output rows [xo0, xo0+NO) of a warp need the source rows xo0-w-pad .. xo0+NO-1+w, processed 4 at a time:
// source row x'+q (q<4) adds khat_{t,a} z_t(x'+q) to output x'+q+a, i.e. to acc[q + ai] of a window that
// starts at output x'-w; after the step the first four window entries are complete and leave.
// PDK >= 1: polynomial basis of total degree PDK (terms t(i,j), i outer: f_i(x) = u_x^i on the spectrum of image j).  The
// terms are grouped by image, c_{j,a}(x') = sum_i khat_{(i,j),a} u_x'^i is formed per source row (f_0 = 1 costs nothing)
// and ONE complex multiply-add per (image, tap, row) follows: 72 instead of 96 FMA per row and tap at DK = 2.
// PDK = -1: any basis, one complex multiply-add per (term, tap, row) on the pre-weighted rows.
// GEN = false: H a power of two (source rows wrap by mask), Nh a multiple of 32.  GEN = true: any H and Nh - rows wrap
// by modulo, columns past the end repeat the last one and store nothing, and the x-range of a warp need not be a
// multiple of 4 (the last group stores its live rows only).  A template parameter: the general tests cost the
// power-of-two kernel 16 registers and 4 % otherwise.
template <int L, int PDK, bool GEN>
__global__ void __launch_bounds__(kFirCols *kFirWarps, 2)
k_fir_x(const double2 *__restrict__ rhat, const double *__restrict__ xwt, const Seq *__restrict__ seqs,
        const double2 *__restrict__ khat, double2 *mhat, FirDims d) {
    constexpr int w = (L - 1) / 2, NA = L + 3;
    extern __shared__ double2 smf[];
    double2 *kh = smf;                                   // [L*FK][32]
    double2 *rt = smf + (size_t)L * d.FK * kFirCols;     // [2][warp][nKa][4][32]
    __shared__ Seq sseq[kFirMaxFK];
    const int tid = threadIdx.x, col = tid & 31, wq = tid >> 5, bz = blockIdx.z;
    const int H = d.H, Nh = d.Nh, FK = d.FK, nKa = d.nKa;
    const int mreal = blockIdx.x * kFirCols + col, m = GEN ? min(mreal, Nh - 1) : mreal;
    const bool packed = (m == 0);          // column 0 holds (X[0], X[W/2]), both real
    for (int i = tid; i < L * FK * kFirCols; i += kFirCols * kFirWarps)
        kh[i] = __ldg(&khat[((size_t)bz * L * FK + (i >> 5)) * Nh +
                            (GEN ? min(blockIdx.x * kFirCols + (i & 31), Nh - 1) : blockIdx.x * kFirCols + (i & 31))]);
    if (tid < FK) sseq[tid] = seqs[tid];
    __syncthreads();
    const int xo0 = (blockIdx.y * kFirWarps + wq) * d.NO;
    if (xo0 >= H) return;
    const int nout = min(d.NO, H - xo0);
    const int xs0 = xo0 - w - d.pad, lead = (2 * w + d.pad) / 4, ngroups = (GEN ? (nout + 3) / 4 : nout / 4) + lead;
    const double2 *rb = rhat + (size_t)bz * d.nimg * H * Nh + m;
    double2 *out = mhat + (size_t)bz * d.nimg * H * Nh + m;               // slot nKa of the spectrum stack
    double2 *rtw = rt + (size_t)wq * nKa * 4 * kFirCols + col;
    const size_t bufstride = (size_t)kFirWarps * nKa * 4 * kFirCols;

    // x-weights f_i(x) of the 4 rows of a group, per warp: lane (i*4+q) fetches one value a group ahead
    // (register), stores it at the top of the next group; __syncwarp orders the store before the reads.
    double *fws = reinterpret_cast<double *>(smf + (size_t)L * FK * kFirCols + 2 * bufstride) + wq * 2 * 4 * kFirMaxNKa;
    const int lane = col;
    auto fetch_w = [&](int g) -> double {
        return lane < nKa * 4 ? __ldg(&xwt[(size_t)(lane >> 2) * H + (GEN ? wrap_index(xs0 + 4 * g + (lane & 3), H, -1) : ((xs0 + 4 * g + (lane & 3)) & (H - 1)))]) : 0.0;
    };
    auto issue = [&](int g) {
        double2 *dst = rtw + (size_t)(g & 1) * bufstride;
        for (int j = 0; j < nKa; ++j)
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int x = GEN ? wrap_index(xs0 + 4 * g + q, H, -1) : ((xs0 + 4 * g + q) & (H - 1));
                cp_async16(dst + (j * 4 + q) * kFirCols, rb + ((size_t)j * H + x) * Nh);
            }
        cp_async_commit();
    };

    double2 acc[NA];
#pragma unroll
    for (int i = 0; i < NA; ++i) acc[i] = make_double2(0.0, 0.0);
    issue(0);
    double wnext = fetch_w(0);
    for (int g = 0; g < ngroups; ++g) {
        double *fw = fws + (g & 1) * 4 * kFirMaxNKa;
        if (lane < nKa * 4) fw[lane] = wnext;
        if (g + 1 < ngroups) { issue(g + 1); wnext = fetch_w(g + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
        __syncwarp();
        const double2 *r = rtw + (size_t)(g & 1) * bufstride;
        const int xg = xs0 + 4 * g;
        if constexpr (PDK >= 1) {
#pragma unroll
            for (int j = 0; j <= PDK; ++j) {
                // operands of the four rows: acc.x += c.x p0 + c.y p1, acc.y += c.x p2 + c.y p3 (the packed column 0 is
                // two real filters: no cross terms)
                double pz[4][4], f[PDK][4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const double2 rv = r[(j * 4 + q) * kFirCols];
                    pz[q][0] = rv.x; pz[q][1] = packed ? 0.0 : -rv.y; pz[q][2] = packed ? 0.0 : rv.y; pz[q][3] = packed ? rv.y : rv.x;
#pragma unroll
                    for (int i = 1; i <= PDK - j; ++i) f[i - 1][q] = fw[i * 4 + q];
                }
                const double2 *kp = kh + col;
#pragma unroll
                for (int ai = 0; ai < L; ++ai) {
                    double2 c[4];
                    const double2 k0 = kp[(size_t)(ai * FK + j) * kFirCols];          // t(0, j) = j
#pragma unroll
                    for (int q = 0; q < 4; ++q) c[q] = k0;
#pragma unroll
                    for (int i = 1; i <= PDK - j; ++i) {
                        // t(i, j) = sum_{i' < i} (PDK + 1 - i') + j
                        const double2 k = kp[(size_t)(ai * FK + i * (PDK + 1) - i * (i - 1) / 2 + j) * kFirCols];
#pragma unroll
                        for (int q = 0; q < 4; ++q) { c[q].x = fma(k.x, f[i - 1][q], c[q].x); c[q].y = fma(k.y, f[i - 1][q], c[q].y); }
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        double2 &a = acc[ai + q];
                        a.x = fma(c[q].x, pz[q][0], a.x);
                        a.y = fma(c[q].x, pz[q][2], a.y);
                        a.x = fma(c[q].y, pz[q][1], a.x);
                        a.y = fma(c[q].y, pz[q][3], a.y);
                    }
                }
            }
        } else {
            for (int t = 0; t < FK; ++t) {
                const Seq sq = sseq[t];
                double2 z[4];
    #pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const double f = fw[sq.xw * 4 + q];
                    const double2 rv = r[(sq.img * 4 + q) * kFirCols];
                    z[q] = make_double2(f * rv.x, f * rv.y);
                }
                const double2 *kp = kh + t * kFirCols + col;
    #pragma unroll
                for (int ai = 0; ai < L; ++ai) {
                    const double2 k = kp[(size_t)ai * FK * kFirCols];
                    const double kb = packed ? 0.0 : -k.y, kc = packed ? k.y : k.x, kd = packed ? 0.0 : k.y;
    #pragma unroll
                    for (int q = 0; q < 4; ++q) cmac(acc[ai + q], k.x, kb, kc, kd, z[q]);
                }
            }
        }
        if (g >= lead) {
            const int xe = xg - w;
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (!GEN || (xe + q < xo0 + nout && mreal < Nh)) out[(size_t)(xe + q) * Nh] = acc[q];
        }
#pragma unroll
        for (int i = 0; i + 4 < NA; ++i) acc[i] = acc[i + 4];
#pragma unroll
        for (int i = NA - 4; i < NA; ++i) acc[i] = make_double2(0.0, 0.0);
    }
}

// D(x, .) = S(x, .) - irfft(mdl(x, .)) - sum_s b_s f'_i(x) g'_j(.)   for one row per thread row.
// The half spectrum X[0..NH) (DC/Nyquist packed in slot 0) is folded back to the NH-point spectrum
// Z = E + i O of z[n] = a[2n] + i a[2n+1]  (E = (X[k] + conj X[NH-k])/2, O = (X[k] - conj X[NH-k]) conj(w^k)/2),
// and the inverse transform is run as conj(FFT(conj Z))/NH on the forward passes.
// grid: x = row group, y = batch; block: (NH/16, RPC).
template <int NH>
__global__ void __launch_bounds__(FftCfg<NH>::T * (FftCfg<NH>::T >= 128 ? 1 : 128 / FftCfg<NH>::T))
k_rowfft_inverse_sub(const double2 *__restrict__ mhat, const double *__restrict__ S, double *__restrict__ D,
                     const double *__restrict__ coef, const double *__restrict__ xwt, const double *__restrict__ gB,
                     const int *__restrict__ bti, const int *__restrict__ btj, const double2 *__restrict__ twW,
                     int H, int nimg, int nKa, int nBa, int FB, int n, int poly) {
    using C = FftCfg<NH>;
    constexpr int T = C::T, RPC = T >= 128 ? 1 : 128 / T, W = 2 * NH;
    extern __shared__ double2 sm2[];
    __shared__ double cj[RPC][16];
    double2 *tw2 = sm2, *buf = sm2 + C::TW2 + threadIdx.y * C::BUF;
    // (H need not be a multiple of RPC: a row slot past the end works on the last row again and stores nothing)
    const int tid = threadIdx.x, xslot = blockIdx.x * RPC + threadIdx.y, x = min(xslot, H - 1), bz = blockIdx.y;
    if (threadIdx.y == 0) fft_load_tw2<NH>(tw2, twW);
    if (tid < nBa) {                 // background of this row as nBa coefficients of the y-basis
        const double *cb = coef + (size_t)bz * n + (n - FB);
        double s = 0.0;
        for (int q = 0; q < FB; ++q)
            if (btj[q] == tid) s = fma(cb[q], __ldg(&xwt[(size_t)(nKa + bti[q]) * H + x]), s);
        cj[threadIdx.y][tid] = s;
    }
    const double2 *X = mhat + ((size_t)bz * nimg * H + x) * NH;
    {
        // the row of S is only needed in the epilogue: pull it towards L2 now (one request per 128-byte line), so that
        // its latency is not exposed a second time after the transform
        const double2 *Sp = reinterpret_cast<const double2 *>(S + ((size_t)bz * H + x) * W);
        if ((tid & 7) == 0) {
#pragma unroll
            for (int r = 0; r < 16; ++r) asm volatile("prefetch.global.L2 [%0];" ::"l"(Sp + tid + r * T));
        }
    }
    double2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int k = tid + r * T;
        const double2 xk = __ldg(&X[k]);
        if (k == 0) {
            v[r] = make_double2(0.5 * (xk.x + xk.y), -0.5 * (xk.x - xk.y));           // conj(E + iO), E, O real
        } else {
            const double2 xn = __ldg(&X[NH - k]), tw = __ldg(&twW[k]);
            const double2 E = make_double2(0.5 * (xk.x + xn.x), 0.5 * (xk.y - xn.y));
            const double2 Dm = make_double2(0.5 * (xk.x - xn.x), 0.5 * (xk.y + xn.y));
            const double2 O = make_double2(Dm.x * tw.x + Dm.y * tw.y, Dm.y * tw.x - Dm.x * tw.y);   // Dm * conj(tw)
            v[r] = make_double2(E.x - O.y, -(E.y + O.x));                               // conj(E + iO)
        }
    }
    __syncthreads();
    fft_core<NH>(v, buf, tw2, twW);
    const size_t o = ((size_t)bz * H + x) * W;
    const double2 *Sr = reinterpret_cast<const double2 *>(S + o);
    double2 *Dr = reinterpret_cast<double2 *>(D + o);
    constexpr double inv = 1.0 / NH;
#pragma unroll 4
    for (int r = 0; r < 16; ++r) {
        const int nn = tid + r * T;
        const double2 zz = buf[nn], sv = Sr[nn];
        double b0 = 0.0, b1 = 0.0;
        if (poly) {      // g'_j(y) = u_y^j, u_y = (2y+1)/W - 1 exact: Horner in registers instead of nBa table reads
            constexpr double invW = 1.0 / W;
            const double u0 = (double)(4 * nn + 1) * invW - 1.0, u1 = (double)(4 * nn + 3) * invW - 1.0;
            for (int j = nBa - 1; j >= 0; --j) {
                const double c = cj[threadIdx.y][j];
                b0 = fma(b0, u0, c);
                b1 = fma(b1, u1, c);
            }
        } else {
            for (int j = 0; j < nBa; ++j) {
                const double2 g = __ldg(reinterpret_cast<const double2 *>(gB + (size_t)j * W) + nn);
                const double c = cj[threadIdx.y][j];
                b0 = fma(c, g.x, b0);
                b1 = fma(c, g.y, b1);
            }
        }
        if (xslot < H) Dr[nn] = make_double2(sv.x - zz.x * inv - b0, sv.y + zz.y * inv - b1);
    }
}

// The same for W not a power of two (W even): the N = W/2 point inverse transform is conj(DFT_N(conj Z)) / N with the
// DFT run as a chirp-z (Bluestein) transform on two M-point register FFTs, exactly as in k_rowfft_forward_bs
// (rowfft.cu): DFT_N(v)[k] = c[k] conv[k], conv = IFFT_M(FFT_M(v c) * bhat).  One CTA of M/16 threads per row.
template <int M>
__global__ void __launch_bounds__(FftCfg<M>::T)
k_rowfft_inverse_sub_bs(const double2 *__restrict__ mhat, const double *__restrict__ S, double *__restrict__ D,
                        const double *__restrict__ coef, const double *__restrict__ xwt, const double *__restrict__ gB,
                        const int *__restrict__ bti, const int *__restrict__ btj, const double2 *__restrict__ twW,
                        const double2 *__restrict__ twM, const double2 *__restrict__ chirp, const double2 *__restrict__ bhat,
                        int H, int W, int nimg, int nKa, int nBa, int FB, int n) {
    using C = FftCfg<M>;
    constexpr int T = C::T;
    extern __shared__ double2 sm4[];
    __shared__ double cj[16];
    double2 *tw2 = sm4, *buf = sm4 + C::TW2;
    const int tid = threadIdx.x, x = blockIdx.x, bz = blockIdx.y, N = W / 2;
    fft_load_tw2<M>(tw2, twM);
    if (tid < nBa) {                 // background of this row as nBa coefficients of the y-basis
        const double *cb = coef + (size_t)bz * n + (n - FB);
        double s = 0.0;
        for (int q = 0; q < FB; ++q)
            if (btj[q] == tid) s = fma(cb[q], __ldg(&xwt[(size_t)(nKa + bti[q]) * H + x]), s);
        cj[tid] = s;
    }
    const double2 *X = mhat + ((size_t)bz * nimg * H + x) * N;
    double2 v[16];
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int k = tid + r * T;
        v[r] = make_double2(0.0, 0.0);
        if (k < N) {
            const double2 xk = __ldg(&X[k]);
            double2 z;
            if (k == 0) {
                z = make_double2(0.5 * (xk.x + xk.y), -0.5 * (xk.x - xk.y));           // conj(E + iO), E, O real
            } else {
                const double2 xn = __ldg(&X[N - k]), tw = __ldg(&twW[k]);
                const double2 E = make_double2(0.5 * (xk.x + xn.x), 0.5 * (xk.y - xn.y));
                const double2 Dm = make_double2(0.5 * (xk.x - xn.x), 0.5 * (xk.y + xn.y));
                const double2 O = make_double2(Dm.x * tw.x + Dm.y * tw.y, Dm.y * tw.x - Dm.x * tw.y);   // Dm * conj(tw)
                z = make_double2(E.x - O.y, -(E.y + O.x));                               // conj(E + iO)
            }
            v[r] = cmulf(z, __ldg(&chirp[k]));
        }
    }
    __syncthreads();                                                       // tw2, cj visible
    fft_core<M>(v, buf, tw2, twM);
#pragma unroll
    for (int r = 0; r < 16; ++r) {
        const int k = tid + r * T;
        const double2 t = cmulf(buf[k], __ldg(&bhat[k]));
        v[r] = make_double2(t.x, -t.y);
    }
    __syncthreads();                                                       // buf consumed before it is rewritten
    fft_core<M>(v, buf, tw2, twM);
    const size_t o = ((size_t)bz * H + x) * W;
    const double2 *Sr = reinterpret_cast<const double2 *>(S + o);
    double2 *Dr = reinterpret_cast<double2 *>(D + o);
    const double inv = 1.0 / ((double)M * (double)N);
    for (int nn = tid; nn < N; nn += T) {
        const double2 u = buf[nn];
        const double2 y = cmulf(make_double2(u.x, -u.y), __ldg(&chirp[nn]));           // M * DFT_N(v)[nn]
        const double2 sv = Sr[nn];
        double b0 = 0.0, b1 = 0.0;
        for (int j = 0; j < nBa; ++j) {
            const double2 g = __ldg(reinterpret_cast<const double2 *>(gB + (size_t)j * W) + nn);
            b0 = fma(cj[j], g.x, b0);
            b1 = fma(cj[j], g.y, b1);
        }
        Dr[nn] = make_double2(sv.x - y.x * inv - b0, sv.y + y.y * inv - b1);             // z = conj(y) / (M N)
    }
}

template <int M>
cudaError_t launch_inv_bs(sfft_plan *p, const double *d_coef, const double *dS, double *dD) {
    using C = FftCfg<M>;
    const size_t smem = (size_t)(C::TW2 + C::BUF) * sizeof(double2);
    auto kern = k_rowfft_inverse_sub_bs<M>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<dim3(p->H, p->nbatch), C::T, smem, p->stream>>>(
        p->rhat + (size_t)p->nKa * p->H * p->Nh, dS, dD, d_coef, p->dt.xwt, p->dt.gB, p->dt.bti, p->dt.btj, p->dt.twW, p->dt.twM,
        p->dt.chirp, p->dt.bhat, p->H, p->W, p->nimg, p->nKa, p->nBa, p->FB, p->n);
    p->launches++;
    return cudaGetLastError();
}

template <int NH>
cudaError_t launch_inv(sfft_plan *p, const double *d_coef, const double *dS, double *dD) {
    using C = FftCfg<NH>;
    constexpr int T = C::T, RPC = T >= 128 ? 1 : 128 / T;
    const size_t smem = (size_t)(C::TW2 + RPC * C::BUF) * sizeof(double2);
    auto kern = k_rowfft_inverse_sub<NH>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<dim3((p->H + RPC - 1) / RPC, p->nbatch), dim3(T, RPC), smem, p->stream>>>(
        p->rhat + (size_t)p->nKa * p->H * p->Nh, dS, dD, d_coef, p->dt.xwt, p->dt.gB, p->dt.bti, p->dt.btj, p->dt.twW,
        p->H, p->nimg, p->nKa, p->nBa, p->FB, p->n, p->basis == SFFT_BASIS_POLY);
    p->launches++;
    return cudaGetLastError();
}

size_t fir_smem(const sfft_plan *p) {
    return ((size_t)p->L * p->FK * kFirCols + 2 * (size_t)kFirWarps * p->nKa * 4 * kFirCols) * sizeof(double2) +
           (size_t)kFirWarps * 2 * 4 * kFirMaxNKa * sizeof(double);
}

template <int L, int PDK, bool GEN>
cudaError_t launch_fir_k2(sfft_plan *p, const FirDims &d, int ny) {
    auto kern = k_fir_x<L, PDK, GEN>;
    const size_t smem = fir_smem(p);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<dim3((p->Nh + kFirCols - 1) / kFirCols, ny, p->nbatch), kFirCols * kFirWarps, smem, p->stream>>>(
        p->rhat, p->dt.xwt, p->dt.seqs, p->khat, p->rhat + (size_t)p->nKa * p->H * p->Nh, d);
    p->launches++;
    return cudaGetLastError();
}

template <int L, int PDK>
cudaError_t launch_fir_k(sfft_plan *p, const FirDims &d, int ny) {
    const bool simple = (p->H & (p->H - 1)) == 0 && p->Nh % kFirCols == 0;
    return simple ? launch_fir_k2<L, PDK, false>(p, d, ny) : launch_fir_k2<L, PDK, true>(p, d, ny);
}

template <int L>
cudaError_t launch_fir(sfft_plan *p, const FirDims &d, int ny) {
    // the grouped form needs the plan's polynomial term order (seqs[t] = (image j, x-power i), i outer)
    if (p->basis == SFFT_BASIS_POLY && p->DK == 1) return launch_fir_k<L, 1>(p, d, ny);
    if (p->basis == SFFT_BASIS_POLY && p->DK == 2) return launch_fir_k<L, 2>(p, d, ny);
    return launch_fir_k<L, -1>(p, d, ny);
}

}  // namespace

// The Fourier route is taken when the row FFT kernels cover W (>= 1024), the FIR kernel is instantiated
// for L, its tables fit in shared memory, and its FP64 work (4 L FK FMA per spectrum point = 2 L FK per
// pixel, plus the transforms, on the plain FMA pipe at ~half the efficiency of the tensor-core contraction)
// is below the direct form's (L+7) * KP tensor-core MACs per pixel.
bool subtract_use_fourier(const sfft_plan *p) {
    if (p->Nh < 512 || p->L < 9 || p->L > 25 || p->FK > kFirMaxFK || p->nKa > kFirMaxNKa || p->nBa > 16) return false;
    if (fir_smem(p) > 200 * 1024) return false;
    const double direct = (double)(p->L + 7) * subtract_kpad(p->nKa, p->L);
    const double fourier = 2.5 * (2.0 * p->L * p->FK) + 40.0 * (p->nKa + 1);
    return fourier < direct;
}

cudaError_t launch_subtract_fourier(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD) {
    const int w = p->w;
    // pixel kernels (Eqs. 3-4) and their row spectra
    cudaError_t e = launch_fold_coef(p, d_coef);
    if (e != cudaSuccess) return e;
    k_kernel_spectrum<<<dim3((p->Nh + 127) / 128, p->L * p->FK, p->nbatch), 128, 0, p->stream>>>(p->kfold, p->dt.twW, p->khat,
                                                                                              p->Nh, p->L, p->FK);
    p->launches++;
    // row spectra of g_j R: transformed again unless the caller promised that this R is the one the last
    // build transformed (sfft_plan_set_reuse_spectra), or the call comes from sfft_run_host* (same staged pair)
    if (!((p->reuse_spectra || p->host_call) && p->rhat_from_build)) {
        e = launch_rowfft_forward(p, dR, nullptr);
        if (e != cudaSuccess) return e;
        p->rhat_from_build = false;
    }
    prof_mark(p, 9);
    // x-ranges: whole waves of 2 CTAs per SM, each warp pays a halo of 2w + pad source rows
    FirDims d{p->H, p->Nh, p->nimg, p->nKa, p->FK, 0, (4 - (2 * w) % 4) % 4};
    const int ncb = (p->Nh + kFirCols - 1) / kFirCols * p->nbatch;
    double best = 1e300; int bny = 1;
    for (int ny = 1; ny <= 64; ++ny) {
        int NO = ((p->H + kFirWarps * ny - 1) / (kFirWarps * ny) + 3) / 4 * 4;
        if (NO < 16) break;
        double cost = ceil((double)ncb * ny / (2.0 * 148.0)) * (NO + 2 * w + d.pad);
        if (cost < best) { best = cost; bny = ny; d.NO = NO; }
    }
    switch (p->L) {
#define SFFT_FIR_CASE(LV) case LV: e = launch_fir<LV>(p, d, bny); break;
        SFFT_FIR_CASE(9) SFFT_FIR_CASE(11) SFFT_FIR_CASE(13) SFFT_FIR_CASE(15) SFFT_FIR_CASE(17)
        SFFT_FIR_CASE(19) SFFT_FIR_CASE(21) SFFT_FIR_CASE(23) SFFT_FIR_CASE(25)
#undef SFFT_FIR_CASE
        default: return cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) return e;
    prof_mark(p, 11);       // FIR done, inverse row transforms next
    switch (p->bsM) {
        case 0: break;
        case 2048: return launch_inv_bs<2048>(p, d_coef, dS, dD);
        case 4096: return launch_inv_bs<4096>(p, d_coef, dS, dD);
        default: return cudaErrorInvalidValue;
    }
    switch (p->Nh) {
        case 512: return launch_inv<512>(p, d_coef, dS, dD);
        case 1024: return launch_inv<1024>(p, d_coef, dS, dD);
        case 2048: return launch_inv<2048>(p, d_coef, dS, dD);
        case 4096: return launch_inv<4096>(p, d_coef, dS, dD);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace sfft
