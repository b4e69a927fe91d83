// Steps a7+a8: spatially varying convolution of the reference by the fitted kernel and the
// difference image (Eqs. 1, 12), fused in one pass over the image:
//   D(x,y) = S(x,y) - sum_{a,b} sum_t k_{t,ab} T_t(x-a,y-b) R(x-a,y-b) - sum_s b_s T'_s(x,y)
// (weights evaluated at the SOURCE pixel: the paper's "weights inside the convolution",
// Eq. 11 / App. A), all indices circular.  With T_t = f_i(x) g_j(y) the x-factor folds into a
// per-source-row kernel  C_j(x'; a,b) = sum_{t:(i,j)} k_{t,ab} f_i(x'),  so the inner loop is
// (number of y-functions) FMAs per kernel tap instead of F_K:
//   D(x,y) = S - sum_j sum_{a,b} C_j(x-a; a,b) * [g_j(y-b) R(x-a,y-b)] - background
//
// k_fold_coef : delta-basis coefficients -> pixel kernels (Eqs. 3-4: centre = a_00 - sum others)
// k_coef_rows : C_j(x'; a,b) for every source row (L2-resident table)
// k_subtract  : one warp owns 4 output rows x 128 columns; per source row it loads a (4+LT-1)-wide
//               register window per lane and reuses it for all rows/taps (FP64-FMA bound).
#include <algorithm>

#include "sfft_internal.h"

namespace sfft {
namespace {

__global__ void k_fold_coef(const double *__restrict__ coef, double *__restrict__ kfold, int n, int FK, int LL) {
    const int t = blockIdx.x, b = blockIdx.y, a0 = LL / 2;
    const double *c = coef + (size_t)b * n + (size_t)t * LL;
    double *k = kfold + ((size_t)b * FK + t) * LL;
    __shared__ double red[32];
    double s = 0.0;
    for (int a = threadIdx.x; a < LL; a += blockDim.x)
        if (a != a0) { double v = c[a]; k[a] = v; s += v; }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int q = 0; q < (int)(blockDim.x >> 5); ++q) tot += red[q];
        k[a0] = c[a0] - tot;
    }
}

// ctab[b][x'][j][ai][bi] (LT x LTP, zero padded around the L x L taps, centred)
__global__ void k_coef_rows(const double *__restrict__ kfold, const double *__restrict__ xwt,
                            const int *__restrict__ kti, const int *__restrict__ ktj, double *__restrict__ ctab,
                            int H, int nKa, int FK, int L, int LT, int LTP) {
    const int x = blockIdx.x, b = blockIdx.y, LL = L * L, off = (LT - L) / 2;
    double *dst = ctab + ((size_t)b * H + x) * nKa * LT * LTP;
    const double *kf = kfold + (size_t)b * FK * LL;
    for (int i = threadIdx.x; i < nKa * LT * LTP; i += blockDim.x) {
        int bi = i % LTP, ai = (i / LTP) % LT, j = i / (LTP * LT);
        int al = ai - off, be = bi - off;
        double v = 0.0;
        if (al >= 0 && al < L && be >= 0 && be < L)
            for (int t = 0; t < FK; ++t)
                if (ktj[t] == j) v = fma(kf[(size_t)t * LL + al * L + be], xwt[(size_t)kti[t] * H + x], v);
        dst[i] = v;
    }
}

constexpr int QX = 4, QY = 4, TY = 128, WARPS = 8, TXR = QX * WARPS;   // CTA tile: 32 rows x 128 columns

template <int LT>
__global__ void __launch_bounds__(32 * WARPS) k_subtract(const double *__restrict__ R, const double *__restrict__ S,
                                                        double *__restrict__ D, const double *__restrict__ ctab,
                                                        const double *__restrict__ coef, const double *__restrict__ gK,
                                                        const double *__restrict__ xwt, const double *__restrict__ gB,
                                                        const int *__restrict__ bti, const int *__restrict__ btj,
                                                        int H, int W, int nKa, int FB, int n, int nKaRows) {
    constexpr int WT = (LT - 1) / 2, LTP = LT + 1, SROWS = TXR + LT - 1, SCOLS = TY + LT + 1, WIN = QY + LT - 1;   // SCOLS even: 16-byte aligned rows
    extern __shared__ double sm[];
    double *Rs = sm;                    // [SROWS][SCOLS] raw reference tile with halo (circular)
    double *gs = sm + SROWS * SCOLS;    // [nKa][SCOLS]   y-weights of the tile's source columns
    const int b = blockIdx.z, x0 = blockIdx.y * TXR, y0 = blockIdx.x * TY;
    const double *Rb = R + (size_t)b * H * W;
    for (int i = threadIdx.x; i < SROWS * SCOLS; i += blockDim.x) {
        int r = i / SCOLS, c = i % SCOLS;
        Rs[i] = __ldg(&Rb[(size_t)((x0 + r - WT) & (H - 1)) * W + ((y0 + c - WT) & (W - 1))]);
    }
    for (int i = threadIdx.x; i < nKa * SCOLS; i += blockDim.x) {
        int j = i / SCOLS, c = i % SCOLS;
        gs[i] = __ldg(&gK[(size_t)j * W + ((y0 + c - WT) & (W - 1))]);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int xr = warp * QX, yc = lane * QY;     // first output row / column of this thread inside the tile
    double acc[QX][QY];
#pragma unroll
    for (int a = 0; a < QX; ++a)
#pragma unroll
        for (int q = 0; q < QY; ++q) acc[a][q] = 0.0;

    // source rows of this warp: tile rows xr .. xr+QX-1+2*WT (tile row r <-> image row x0 + r - WT)
    for (int sr = 0; sr < QX + LT - 1; ++sr) {
        const int trow = xr + sr;
        const int xsrc = (x0 + trow - WT) & (H - 1);
        double wraw[WIN];
#pragma unroll
        for (int q = 0; q < WIN / 2; ++q) {
            double2 t2 = *reinterpret_cast<const double2 *>(&Rs[trow * SCOLS + yc + 2 * q]);
            wraw[2 * q] = t2.x; wraw[2 * q + 1] = t2.y;
        }
        const double *crow = ctab + ((size_t)b * H + xsrc) * nKa * LT * LTP;
        for (int j = 0; j < nKa; ++j) {
            double v[WIN];
#pragma unroll
            for (int q = 0; q < WIN / 2; ++q) {
                double2 g2 = *reinterpret_cast<const double2 *>(&gs[j * SCOLS + yc + 2 * q]);
                v[2 * q] = wraw[2 * q] * g2.x; v[2 * q + 1] = wraw[2 * q + 1] * g2.y;
            }
#pragma unroll
            for (int a = 0; a < QX; ++a) {
                // output row (xr + a) reads source tile row (xr + a - alpha + WT) => alpha index ai = a + LT-1 - sr
                const int ai = a + LT - 1 - sr;
                if (ai >= 0 && ai < LT) {
                    const double *cr = crow + ((size_t)j * LT + ai) * LTP;
#pragma unroll
                    for (int b2 = 0; b2 < LTP / 2; ++b2) {
                        // tap beta index bi reads source column y - beta = yc + q + (LT-1-bi) in window coordinates
                        const double2 c2 = __ldg(reinterpret_cast<const double2 *>(cr) + b2);
#pragma unroll
                        for (int q = 0; q < QY; ++q) acc[a][q] = fma(c2.x, v[q + LT - 1 - 2 * b2], acc[a][q]);
                        if (2 * b2 + 1 < LT) {
#pragma unroll
                            for (int q = 0; q < QY; ++q) acc[a][q] = fma(c2.y, v[q + LT - 2 - 2 * b2], acc[a][q]);
                        }
                    }
                }
            }
        }
    }
    const double *cb = coef + (size_t)b * n + (n - FB);
#pragma unroll
    for (int a = 0; a < QX; ++a) {
        const int x = x0 + xr + a;
        if (x >= H) continue;
#pragma unroll
        for (int q = 0; q < QY; ++q) {
            const int y = y0 + yc + q;
            if (y >= W) continue;
            double bg = 0.0;
            for (int s = 0; s < FB; ++s)
                bg = fma(cb[s] * __ldg(&xwt[(size_t)(nKaRows + bti[s]) * H + x]), __ldg(&gB[(size_t)btj[s] * W + y]), bg);
            const size_t o = ((size_t)b * H + x) * W + y;
            D[o] = S[o] - acc[a][q] - bg;
        }
    }
}

template <int LT>
cudaError_t launch_sub(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD) {
    constexpr int SROWS = TXR + LT - 1, SCOLS = TY + LT + 1;
    size_t smem = (size_t)(SROWS * SCOLS + p->nKa * SCOLS) * sizeof(double);
    auto kern = k_subtract<LT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((p->W + TY - 1) / TY, (p->H + TXR - 1) / TXR, p->nbatch);
    kern<<<grid, 32 * WARPS, smem, p->stream>>>(dR, dS, dD, p->ctab, d_coef, p->dt.gK, p->dt.xwt, p->dt.gB, p->dt.bti,
                                               p->dt.btj, p->H, p->W, p->nKa, p->FB, p->n, p->nKa);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace

int subtract_tap_width(int L) {
    const int sizes[] = {3, 7, 11, 15, 17, 21, 25, 33};
    for (int s : sizes) if (s >= L) return s;
    return 33;
}

cudaError_t launch_subtract(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD) {
    const int LL = p->L * p->L, LT = p->LT, LTP = LT + 1;
    k_fold_coef<<<dim3(p->FK, p->nbatch), 128, 0, p->stream>>>(d_coef, p->kfold, p->n, p->FK, LL);
    k_coef_rows<<<dim3(p->H, p->nbatch), 256, 0, p->stream>>>(p->kfold, p->dt.xwt, p->dt.kti, p->dt.ktj, p->ctab, p->H,
                                                             p->nKa, p->FK, p->L, LT, LTP);
    p->launches += 2;
    prof_mark(p, 9);
    switch (LT) {
        case 3: return launch_sub<3>(p, d_coef, dR, dS, dD);
        case 7: return launch_sub<7>(p, d_coef, dR, dS, dD);
        case 11: return launch_sub<11>(p, d_coef, dR, dS, dD);
        case 15: return launch_sub<15>(p, d_coef, dR, dS, dD);
        case 17: return launch_sub<17>(p, d_coef, dR, dS, dD);
        case 21: return launch_sub<21>(p, d_coef, dR, dS, dD);
        case 25: return launch_sub<25>(p, d_coef, dR, dS, dD);
        case 33: return launch_sub<33>(p, d_coef, dR, dS, dD);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace sfft
