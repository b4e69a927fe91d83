// NEXT-3: noise decorrelation of the difference image (App. C; readings DESIGN g22).
//   Q0^ = sqrt( sigma_D^2 / { sum_j s2_Sj |G_j^|^2 + sum_i s2_Ri |K^|^2 |H_i^|^2 } )          (C20)
// with the unit-kernel-sum normalisation of PAPER.md:627 (sigma_D^2 = the denominator at zero frequency), applied
// segment by segment: the image is cut in square tiles of T pixels, in each tile the fitted,
// spatially varying kernel is frozen at the tile's centre pixel, and the tile is convolved circularly with Q.
//
// Three passes over the image, all transforms in shared memory (T <= 512):
//   k_seg_forward : every image row is W/T independent real T-point segments -> half spectra (y direction)
//   k_tile_cols   : per tile and group of frequency columns: T-point complex transform along x, multiplication
//                   by Q0^(l,m) (formed on the fly from the tile's kernel and the G/H tables), inverse along x
//   k_seg_inverse : half spectra -> real segments (y direction)
// A real segment of T points is transformed as T/2 complex points + even/odd split, DC and Nyquist packed in
// slot 0, exactly as the full-row transforms of rowfft.cu.
#include "sfft_internal.h"

namespace sfft {
namespace {

__device__ __forceinline__ double2 cmul2(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}

// One Stockham radix-R pass over `nfft` independent N-point transforms stored back to back in shared memory.
// twT[q] = exp(-2 pi i q / TT); N divides TT.
template <int R>
__device__ __forceinline__ void stockham_batched(const double2 *in, double2 *out, int N, int Ns, int nfft, const double2 *twT,
                                                 int TT) {
    const int per = N / R;
    for (int idx = threadIdx.x; idx < nfft * per; idx += blockDim.x) {
        const int f = idx / per, j = idx - f * per, k = j & (Ns - 1);
        const double2 *src = in + f * N;
        double2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = src[j + r * per];
        if (Ns > 1) {
            const int step = (TT / (Ns * R)) * k;
#pragma unroll
            for (int r = 1; r < R; ++r) v[r] = cmul2(v[r], twT[(r * step) & (TT - 1)]);
        }
        double2 *dst = out + f * N + (j - k) * R + k;
        if (R == 4) {
            const double2 t0 = make_double2(v[0].x + v[2].x, v[0].y + v[2].y), t1 = make_double2(v[0].x - v[2].x, v[0].y - v[2].y);
            const double2 t2 = make_double2(v[1].x + v[3].x, v[1].y + v[3].y), d = make_double2(v[1].x - v[3].x, v[1].y - v[3].y);
            const double2 t3 = make_double2(d.y, -d.x);
            dst[0] = make_double2(t0.x + t2.x, t0.y + t2.y);
            dst[Ns] = make_double2(t1.x + t3.x, t1.y + t3.y);
            dst[2 * Ns] = make_double2(t0.x - t2.x, t0.y - t2.y);
            dst[3 * Ns] = make_double2(t1.x - t3.x, t1.y - t3.y);
        } else {
            dst[0] = make_double2(v[0].x + v[1].x, v[0].y + v[1].y);
            dst[Ns] = make_double2(v[0].x - v[1].x, v[0].y - v[1].y);
        }
    }
}

// Forward transforms of `nfft` N-point sequences (N a power of two) held in `a`; returns the buffer with the result.
__device__ __forceinline__ double2 *fft_batched(double2 *a, double2 *b, int N, int nfft, const double2 *twT, int TT) {
    int Ns = 1;
    double2 *in = a, *out = b;
    while (Ns * 4 <= N) {
        stockham_batched<4>(in, out, N, Ns, nfft, twT, TT);
        __syncthreads();
        Ns *= 4;
        double2 *t = in; in = out; out = t;
    }
    if (Ns < N) {
        stockham_batched<2>(in, out, N, Ns, nfft, twT, TT);
        __syncthreads();
        double2 *t = in; in = out; out = t;
    }
    return in;
}

// twT[q] = exp(-2 pi i q / T), q < T  (exact at the octants)
__global__ void k_decorr_twiddles(double2 *twT, int T) {
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= T) return;
    double s, c;
    sincospi(-2.0 * (double)q / (double)T, &s, &c);
    twT[q] = make_double2(c, s);
}

// Tile-independent part of the C20 denominator on the half grid l < T, m <= T/2:
//   sg[l][m] = sum_j varS_j |G_j^(l,m)|^2,  sh[l][m] = sum_i varR_i |H_i^(l,m)|^2,  kernels centred, LG x LG / LH x LH.
__global__ void k_decorr_tables(const double *__restrict__ kern, const double *__restrict__ var, int nk, int Lk,
                                double *__restrict__ out, int T) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, NH1 = T / 2 + 1;
    if (i >= T * NH1) return;
    const int l = i / NH1, m = i - l * NH1, wk = (Lk - 1) / 2;
    double acc = 0.0;
    for (int j = 0; j < nk; ++j) {
        double re = 0.0, im = 0.0;
        for (int a = 0; a < Lk; ++a)
            for (int b = 0; b < Lk; ++b) {
                double s, c;
                sincospi(-2.0 * (double)((l * (a - wk) + m * (b - wk)) % T) / (double)T, &s, &c);
                const double v = kern[((size_t)j * Lk + a) * Lk + b];
                re = fma(v, c, re);
                im = fma(v, s, im);
            }
        acc = fma(var[j], re * re + im * im, acc);
    }
    out[i] = acc;
}

// y direction, forward: one CTA per image row; its W/T segments are transformed together.
// grid: x = row, y = batch.  ahat[b][x][seg*T/2 + k], k < T/2, slot 0 = (X[0], X[T/2]).
__global__ void __launch_bounds__(256) k_seg_forward(const double *__restrict__ D, double2 *__restrict__ ahat,
                                                     const double2 *__restrict__ twg, int H, int W, int T) {
    extern __shared__ double2 smd[];
    const int NHt = T / 2, nseg = W / T, x = blockIdx.x, bz = blockIdx.y;
    double2 *tw = smd, *a = smd + T, *b = a + W / 2;
    for (int i = threadIdx.x; i < T; i += blockDim.x) tw[i] = twg[i];
    const double2 *src = reinterpret_cast<const double2 *>(D + ((size_t)bz * H + x) * W);
    for (int i = threadIdx.x; i < W / 2; i += blockDim.x) a[i] = src[i];           // z[n] = d[2n] + i d[2n+1], segment by segment
    __syncthreads();
    const double2 *Z = fft_batched(a, b, NHt, nseg, tw, T);
    double2 *dst = ahat + ((size_t)bz * H + x) * (W / 2);
    for (int i = threadIdx.x; i < nseg * (NHt / 2 + 1); i += blockDim.x) {
        const int f = i / (NHt / 2 + 1), k = i - f * (NHt / 2 + 1);
        const double2 *z = Z + f * NHt;
        double2 *o = dst + f * NHt;
        if (k == 0) {
            o[0] = make_double2(z[0].x + z[0].y, z[0].x - z[0].y);
        } else {
            const double2 zk = z[k], zn = z[NHt - k];
            const double2 E = make_double2(0.5 * (zk.x + zn.x), 0.5 * (zk.y - zn.y));
            const double2 O = make_double2(0.5 * (zk.y + zn.y), -0.5 * (zk.x - zn.x));
            const double2 wO = cmul2(tw[k], O);
            o[k] = make_double2(E.x + wO.x, E.y + wO.y);
            if (k != NHt - k) o[NHt - k] = make_double2(E.x - wO.x, -(E.y - wO.y));
        }
    }
}

// y direction, inverse: half spectra -> real segments, out = irfft / 1 (the 1/T of the x direction is applied in k_tile_cols).
__global__ void __launch_bounds__(256) k_seg_inverse(const double2 *__restrict__ ahat, double *__restrict__ out,
                                                     const double2 *__restrict__ twg, int H, int W, int T) {
    extern __shared__ double2 smd[];
    const int NHt = T / 2, nseg = W / T, x = blockIdx.x, bz = blockIdx.y;
    double2 *tw = smd, *a = smd + T, *b = a + W / 2;
    for (int i = threadIdx.x; i < T; i += blockDim.x) tw[i] = twg[i];
    __syncthreads();
    const double2 *X = ahat + ((size_t)bz * H + x) * (W / 2);
    for (int i = threadIdx.x; i < W / 2; i += blockDim.x) {
        const int f = i / NHt, k = i - f * NHt;
        const double2 xk = X[i];
        if (k == 0) {
            a[i] = make_double2(0.5 * (xk.x + xk.y), -0.5 * (xk.x - xk.y));            // conj(E + iO), E, O real
        } else {
            const double2 xn = X[f * NHt + NHt - k], t = tw[k];
            const double2 E = make_double2(0.5 * (xk.x + xn.x), 0.5 * (xk.y - xn.y));
            const double2 Dm = make_double2(0.5 * (xk.x - xn.x), 0.5 * (xk.y + xn.y));
            const double2 O = make_double2(Dm.x * t.x + Dm.y * t.y, Dm.y * t.x - Dm.x * t.y);   // Dm * conj(w^k)
            a[i] = make_double2(E.x - O.y, -(E.y + O.x));                                   // conj(E + iO)
        }
    }
    __syncthreads();
    const double2 *Z = fft_batched(a, b, NHt, nseg, tw, T);
    double2 *dst = reinterpret_cast<double2 *>(out + ((size_t)bz * H + x) * W);
    const double inv = 1.0 / NHt;
    for (int i = threadIdx.x; i < W / 2; i += blockDim.x) dst[i] = make_double2(Z[i].x * inv, -Z[i].y * inv);
}

struct TileDims { int H, W, T, L, FK, nKa, MC; };

// x direction: tile (a, b), frequency columns m0 .. m0+MC-1 of the tile's T/2 (slot 0 packs m = 0 and m = T/2).
// grid: x = column group, y = tile index (a * W/T + b), z = batch.
__global__ void __launch_bounds__(256) k_tile_cols(double2 *__restrict__ ahat, const double *__restrict__ kfold,
                                                   const double *__restrict__ xwt, const double *__restrict__ gK,
                                                   const int *__restrict__ kti, const int *__restrict__ ktj,
                                                   const double *__restrict__ sg, const double *__restrict__ sh,
                                                   const double2 *__restrict__ twg, TileDims d) {
    extern __shared__ double2 smd[];
    const int T = d.T, NHt = T / 2, NH1 = NHt + 1, L = d.L, LL = L * L, w = (L - 1) / 2, MC = d.MC;
    const int ntx = d.W / T, ta = blockIdx.y / ntx, tb = blockIdx.y - ta * ntx, bz = blockIdx.z, m0 = blockIdx.x * MC;
    double2 *tw = smd, *a = smd + T, *b = a + MC * T;
    double *Ks = reinterpret_cast<double *>(b + MC * T);            // [L][L] kernel frozen at the tile centre
    double2 *Kb = reinterpret_cast<double2 *>(Ks + LL + (LL & 1));  // [MC + 1][L] partial transforms over beta (extra: m = T/2)
    const int tid = threadIdx.x;
    for (int i = tid; i < T; i += blockDim.x) tw[i] = twg[i];
    const int xc = ta * T + T / 2, yc = tb * T + T / 2;
    for (int i = tid; i < LL; i += blockDim.x) {
        double v = 0.0;
        for (int t = 0; t < d.FK; ++t)
            v = fma(kfold[((size_t)bz * d.FK + t) * LL + i], xwt[(size_t)kti[t] * d.H + xc] * gK[(size_t)ktj[t] * d.W + yc], v);
        Ks[i] = v;
    }
    // load the MC columns of the tile: a[c][x]
    double2 *base = ahat + ((size_t)bz * d.H + (size_t)ta * T) * (d.W / 2) + (size_t)tb * NHt + m0;
    for (int i = tid; i < MC * T; i += blockDim.x) {
        const int x = i / MC, c = i - x * MC;
        a[c * T + x] = base[(size_t)x * (d.W / 2) + c];
    }
    __syncthreads();
    // partial kernel transforms over beta for the columns of this group (and m = T/2 for the packed column)
    for (int i = tid; i < (MC + 1) * L; i += blockDim.x) {
        const int c = i / L, al = i - c * L, m = c < MC ? m0 + c : NHt;
        double re = 0.0, im = 0.0;
        for (int be = 0; be < L; ++be) {
            const double2 e = tw[(m * (be - w)) & (T - 1)];
            const double v = Ks[al * L + be];
            re = fma(v, e.x, re);
            im = fma(v, e.y, im);
        }
        Kb[i] = make_double2(re, im);
    }
    double2 *Z = fft_batched(a, b, T, MC, tw, T);         // (includes the barrier that publishes Kb)
    double2 *other = (Z == a) ? b : a;
    double ksum = 0.0;
    for (int i = 0; i < LL; ++i) ksum += Ks[i];
    const double den0 = sg[0] + ksum * ksum * sh[0];
    auto q0 = [&](int l, int c, int m) {                  // Q0^(l, m) of Eq. C20 with the unit-sum normalisation
        double re = 0.0, im = 0.0;
        for (int al = 0; al < L; ++al) {
            const double2 e = tw[(l * (al - w)) & (T - 1)], k = Kb[c * L + al];
            re += k.x * e.x - k.y * e.y;
            im += k.x * e.y + k.y * e.x;
        }
        const double den = sg[(size_t)l * NH1 + m] + (re * re + im * im) * sh[(size_t)l * NH1 + m];
        return sqrt(den0 / den);
    };
    // multiply, conjugate (inverse transform = conj(FFT(conj .)) / T), into the other buffer
    const double invT = 1.0 / T;
    for (int i = tid; i < MC * T; i += blockDim.x) {
        const int c = i / T, l = i - c * T, m = m0 + c;
        double2 r;
        if (m != 0) {
            const double q = q0(l, c, m) * invT;
            const double2 z = Z[i];
            r = make_double2(z.x * q, -z.y * q);
        } else {
            // packed column: c(x) = dc(x) + i ny(x), both real along x; their transforms are the Hermitian and
            // anti-Hermitian parts of C^; each is scaled by its own (real, even in l) Q0^ row
            const double2 z = Z[i], zn = Z[c * T + ((T - l) & (T - 1))];
            const double2 A = make_double2(0.5 * (z.x + zn.x), 0.5 * (z.y - zn.y));      // DC part
            const double2 Bv = make_double2(0.5 * (z.y + zn.y), -0.5 * (z.x - zn.x));    // Nyquist part
            const double qa = q0(l, c, 0) * invT, qb = q0(l, MC, NHt) * invT;
            const double2 cz = make_double2(A.x * qa - Bv.y * qb, A.y * qa + Bv.x * qb); // A qa + i B qb
            r = make_double2(cz.x, -cz.y);
        }
        other[i] = r;
    }
    __syncthreads();
    double2 *Y = fft_batched(other, Z, T, MC, tw, T);
    for (int i = tid; i < MC * T; i += blockDim.x) {
        const int x = i / MC, c = i - x * MC;
        const double2 y = Y[c * T + x];
        base[(size_t)x * (d.W / 2) + c] = make_double2(y.x, -y.y);
    }
}

}  // namespace

// scratch (spectrum area of the workspace): ahat [nb][H][W/2] double2, twT [T], sg, sh [T][T/2+1], G/H kernels + variances
cudaError_t launch_decorrelate(sfft_plan *p, const double *d_coef, const double *dD, double *dOut, int T, int nS,
                               const double *h_varS, int LG, const double *h_G, int nR, const double *h_varR, int LH,
                               const double *h_H) {
    const int H = p->H, W = p->W, nb = p->nbatch, NH1 = T / 2 + 1;
    const size_t P = (size_t)H * W;
    double2 *ahat = p->rhat;
    double2 *twT = ahat + (size_t)nb * P / 2;
    double *sg = reinterpret_cast<double *>(twT + T), *sh = sg + (size_t)T * NH1;
    double *dG = sh + (size_t)T * NH1, *dvS = dG + (size_t)nS * LG * LG, *dH = dvS + nS, *dvR = dH + (size_t)nR * LH * LH;
    // The caller's tables (a few KB, laid out on the device as G, varS, H, varR back to back) are copied into a buffer
    // the plan owns and uploaded from there: with page-locked caller arrays an asynchronous copy would still be reading
    // them after this call has returned, and the header promises they are free again by then.  The previous call's
    // upload may still be reading that buffer: wait for the stream before overwriting it.
    const size_t nG = (size_t)nS * LG * LG, nH = (size_t)nR * LH * LH, ntab = nG + nS + nH + nR;
    cudaError_t e = p->decorr_host.empty() ? cudaSuccess : cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return e;
    p->decorr_host.resize(ntab);
    std::copy(h_G, h_G + nG, p->decorr_host.begin());
    std::copy(h_varS, h_varS + nS, p->decorr_host.begin() + nG);
    std::copy(h_H, h_H + nH, p->decorr_host.begin() + nG + nS);
    std::copy(h_varR, h_varR + nR, p->decorr_host.begin() + nG + nS + nH);
    e = cudaMemcpyAsync(dG, p->decorr_host.data(), sizeof(double) * ntab, cudaMemcpyHostToDevice, p->stream);
    if (e != cudaSuccess) return e;
    e = launch_fold_coef(p, d_coef);                      // pixel kernels of Eqs. 3-4 (kfold)
    if (e != cudaSuccess) return e;
    k_decorr_twiddles<<<(T + 127) / 128, 128, 0, p->stream>>>(twT, T);
    k_decorr_tables<<<(T * NH1 + 127) / 128, 128, 0, p->stream>>>(dG, dvS, nS, LG, sg, T);
    k_decorr_tables<<<(T * NH1 + 127) / 128, 128, 0, p->stream>>>(dH, dvR, nR, LH, sh, T);
    const size_t smem_seg = (size_t)(T + W) * sizeof(double2);
    e = cudaFuncSetAttribute(k_seg_forward, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_seg);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_seg_inverse, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_seg);
    if (e != cudaSuccess) return e;
    k_seg_forward<<<dim3(H, nb), 256, smem_seg, p->stream>>>(dD, ahat, twT, H, W, T);
    TileDims d{H, W, T, p->L, p->FK, p->nKa, 0};
    d.MC = std::max(1, std::min(T / 2, 4096 / T));
    const int LL = p->L * p->L;
    const size_t smem_tile = (size_t)(T + 2 * d.MC * T) * sizeof(double2) + (size_t)(LL + (LL & 1)) * sizeof(double) +
                             (size_t)(d.MC + 1) * p->L * sizeof(double2);
    e = cudaFuncSetAttribute(k_tile_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_tile);
    if (e != cudaSuccess) return e;
    k_tile_cols<<<dim3((T / 2) / d.MC, (H / T) * (W / T), nb), 256, smem_tile, p->stream>>>(
        ahat, p->kfold, p->dt.xwt, p->dt.gK, p->dt.kti, p->dt.ktj, sg, sh, twT, d);
    k_seg_inverse<<<dim3(H, nb), 256, smem_seg, p->stream>>>(ahat, dOut, twT, H, W, T);
    p->launches += 6;
    return cudaGetLastError();
}

}  // namespace sfft
