// Steps a7+a8: spatially varying convolution of the reference by the fitted kernel and the
// difference image (Eqs. 1, 12), fused in one pass over the image:
//   D(x,y) = S(x,y) - sum_{a,b} sum_t k_{t,ab} T_t(x-a,y-b) R(x-a,y-b) - sum_s b_s T'_s(x,y)
// (weights evaluated at the SOURCE pixel: the paper's "weights inside the convolution",
// Eq. 11 / App. A), all indices circular.  With T_t = f_i(x) g_j(y) the x-factor folds into a
// per-source-row kernel  C_j(x'; a,b) = sum_{t:(i,j)} k_{t,ab} f_i(x'),  so
//   D(x,y) = S - sum_{x'} sum_{(j,b)} C_j(x'; x-x', b) * V_j(x', y-b) - background,   V_j = g_j R.
//
// For 8 consecutive output rows this is a dense contraction on the FP64 tensor cores
// (mma.sync.m8n8k4.f64): rows = output rows, K = (source row x', (j,b)) over the L+7 source rows
// of the band (coefficient 0 where |x-x'| > w), columns = 8 consecutive y.  The right operand is
// Toeplitz in (b, y): lane (k, n) reads V_j(x', y0 + n - b_k) straight from the staged row, so
// the image is never unfolded.
//
// k_fold_coef : delta-basis coefficients -> pixel kernels (Eqs. 3-4: centre = a_00 - sum others)
// k_coef_rows : ctab[x'][a][(j,b)] = C_j(x'; a, b) for every source row (L2-resident table)
// k_subtract  : CTA = 8 output rows x 64*NBW columns, 8 warps side by side in y, source rows
//               streamed through shared memory RS at a time.
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

// ctab[b][x'][ai][kk], kk = j*L + bi (zero padded to KP)
__global__ void k_coef_rows(const double *__restrict__ kfold, const double *__restrict__ xwt,
                            const int *__restrict__ kti, const int *__restrict__ ktj, double *__restrict__ ctab,
                            int H, int nKa, int FK, int L, int KP) {
    const int x = blockIdx.x, b = blockIdx.y, LL = L * L;
    double *dst = ctab + ((size_t)b * H + x) * L * KP;
    const double *kf = kfold + (size_t)b * FK * LL;
    for (int i = threadIdx.x; i < L * KP; i += blockDim.x) {
        const int kk = i % KP, ai = i / KP, j = kk / L, bi = kk - j * L;
        double v = 0.0;
        if (j < nKa)
            for (int t = 0; t < FK; ++t)
                if (ktj[t] == j) v = fma(kf[(size_t)t * LL + ai * L + bi], xwt[(size_t)kti[t] * H + x], v);
        dst[i] = v;
    }
}

struct SubDims { int H, W, L, w, nKa, FB, n, KP, NKS, PS, ASTR, RS, NSRC, hmask, wmask; };   // masks: N - 1 for powers of two, else -1

// grid: x = column tile (64*NBW), y = 8-row block, z = batch.  block: 256 (warp = 8*NBW columns).
template <int NBW>
__global__ void __launch_bounds__(256) k_subtract(const double *__restrict__ R, const double *__restrict__ S,
                                                  double *__restrict__ D, const double *__restrict__ ctab,
                                                  const double *__restrict__ coef, const double *__restrict__ gK,
                                                  const double *__restrict__ xwt, const double *__restrict__ gB,
                                                  const int *__restrict__ bti, const int *__restrict__ btj, SubDims d) {
    constexpr int TY = 64 * NBW;
    extern __shared__ double sm[];
    double *Vs = sm;                                     // [RS][nKa][PS]   g_j(y) R(x', y) with a w-wide halo
    double *As = sm + (size_t)d.RS * d.nKa * d.PS;       // [RS][8][ASTR]   C_j(x'; x0+r-x', b)
    int *offt = reinterpret_cast<int *>(As + (size_t)d.RS * 8 * d.ASTR);   // [KP] B-fragment offset of K index kk
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, r = lane >> 2, kq = lane & 3;
    const int bz = blockIdx.z, x0 = blockIdx.y * 8, y0 = blockIdx.x * TY;
    const double *Rb = R + (size_t)bz * d.H * d.W;
    const double *ct = ctab + (size_t)bz * d.H * d.L * d.KP;
    const int nvc = TY + d.L - 1;                        // staged columns: y0 - w .. y0 + TY + w - 1
    for (int kk = tid; kk < d.KP; kk += 256) {
        const int kc = min(kk, d.nKa * d.L - 1), j = kc / d.L, bi = kc - j * d.L;
        offt[kk] = j * d.PS + 2 * d.w - bi;              // column (y - y0) + w - beta,  beta = bi - w
    }
    double acc[NBW][2];
#pragma unroll
    for (int nb = 0; nb < NBW; ++nb) acc[nb][0] = acc[nb][1] = 0.0;
    const int wcol = warp * 8 * NBW;

    for (int s0 = 0; s0 < d.NSRC; s0 += d.RS) {
        const int ns = min(d.RS, d.NSRC - s0);
        __syncthreads();
        for (int i = tid; i < ns * nvc; i += 256) {
            const int dd = i / nvc, cs = i - dd * nvc;
            const int xs = wrap_index(x0 - d.w + s0 + dd, d.H, d.hmask), y = wrap_index(y0 - d.w + cs, d.W, d.wmask);
            const double v = __ldg(&Rb[(size_t)xs * d.W + y]);
            for (int j = 0; j < d.nKa; ++j) Vs[((size_t)dd * d.nKa + j) * d.PS + cs] = v * __ldg(&gK[(size_t)j * d.W + y]);
        }
        for (int i = tid; i < ns * 8 * d.KP; i += 256) {
            const int kk = i % d.KP, rr = (i / d.KP) & 7, dd = i / (d.KP * 8);
            const int xs = wrap_index(x0 - d.w + s0 + dd, d.H, d.hmask);
            const int ai = rr + 2 * d.w - (s0 + dd);      // alpha + w,  alpha = (x0 + rr) - (x0 - w + s0 + dd)
            As[((size_t)dd * 8 + rr) * d.ASTR + kk] =
                (ai >= 0 && ai < d.L) ? __ldg(&ct[((size_t)xs * d.L + ai) * d.KP + kk]) : 0.0;
        }
        __syncthreads();
        for (int dd = 0; dd < ns; ++dd) {
            const double *ap = As + ((size_t)dd * 8 + r) * d.ASTR + kq;
            const double *vp = Vs + (size_t)dd * d.nKa * d.PS + wcol + r;
#pragma unroll 2
            for (int ks = 0; ks < d.NKS; ++ks) {
                const double a = ap[4 * ks];
                const double *bp = vp + offt[4 * ks + kq];
#pragma unroll
                for (int nb = 0; nb < NBW; ++nb) dmma884(acc[nb], a, bp[8 * nb]);
            }
        }
    }
    // epilogue: D = S - model - background (the last tiles of a frame that is not a multiple of the tile overhang)
    const int x = x0 + r;
    if (x >= d.H) return;
    const double *cb = coef + (size_t)bz * d.n + (d.n - d.FB);
#pragma unroll
    for (int nb = 0; nb < NBW; ++nb) {
        const int y = y0 + wcol + 8 * nb + 2 * kq;
        if (y >= d.W) continue;                          // W is even: y + 1 < W as well
        double bg0 = 0.0, bg1 = 0.0;
        for (int s = 0; s < d.FB; ++s) {
            const double cf = cb[s] * __ldg(&xwt[(size_t)(d.nKa + bti[s]) * d.H + x]);
            const double *g = gB + (size_t)btj[s] * d.W + y;
            bg0 = fma(cf, __ldg(&g[0]), bg0);
            bg1 = fma(cf, __ldg(&g[1]), bg1);
        }
        const size_t o = ((size_t)bz * d.H + x) * d.W + y;
        const double2 sv = *reinterpret_cast<const double2 *>(&S[o]);
        *reinterpret_cast<double2 *>(&D[o]) = make_double2(sv.x - acc[nb][0] - bg0, sv.y - acc[nb][1] - bg1);
    }
}

template <int NBW>
cudaError_t launch_sub(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD, SubDims d) {
    constexpr int TY = 64 * NBW;
    d.PS = ((TY + d.L - 1 + 7) / 8) * 8 + 8;
    auto bytes = [&](int rs) { return ((size_t)rs * d.nKa * d.PS + (size_t)rs * 8 * d.ASTR) * sizeof(double) + (size_t)d.KP * sizeof(int); };
    d.RS = 4;
    while (d.RS > 1 && bytes(d.RS) > 72 * 1024) d.RS >>= 1;
    const size_t smem = bytes(d.RS);
    auto kern = k_subtract<NBW>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((p->W + TY - 1) / TY, (p->H + 7) / 8, p->nbatch);
    kern<<<grid, 256, smem, p->stream>>>(dR, dS, dD, p->ctab, d_coef, p->dt.gK, p->dt.xwt, p->dt.gB, p->dt.bti, p->dt.btj, d);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_fold_coef(sfft_plan *p, const double *d_coef) {
    k_fold_coef<<<dim3(p->FK, p->nbatch), 128, 0, p->stream>>>(d_coef, p->kfold, p->n, p->FK, p->L * p->L);
    p->launches++;
    return cudaGetLastError();
}

// K extent of one source row of the subtract contraction: nKa*L padded to whole k4 steps
int subtract_kpad(int nKa, int L) { return 4 * ((nKa * L + 3) / 4); }

cudaError_t launch_subtract(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD) {
    if (subtract_use_fourier(p)) return launch_subtract_fourier(p, d_coef, dR, dS, dD);
    SubDims d{};
    d.H = p->H; d.W = p->W; d.L = p->L; d.w = p->w; d.nKa = p->nKa; d.FB = p->FB; d.n = p->n;
    d.KP = subtract_kpad(p->nKa, p->L); d.NKS = d.KP / 4;
    d.ASTR = ((d.KP + 15) / 16) * 16 + 4;
    d.NSRC = p->L + 7;
    d.hmask = (p->H & (p->H - 1)) == 0 ? p->H - 1 : -1;
    d.wmask = (p->W & (p->W - 1)) == 0 ? p->W - 1 : -1;
    cudaError_t e = launch_fold_coef(p, d_coef);
    if (e != cudaSuccess) return e;
    k_coef_rows<<<dim3(p->H, p->nbatch), 256, 0, p->stream>>>(p->kfold, p->dt.xwt, p->dt.kti, p->dt.ktj, p->ctab, p->H,
                                                             p->nKa, p->FK, p->L, d.KP);
    p->launches++;
    prof_mark(p, 9);
    if (p->W >= 512) return launch_sub<8>(p, d_coef, dR, dS, dD, d);
    if (p->W >= 256) return launch_sub<4>(p, d_coef, dR, dS, dD, d);
    if (p->W >= 128) return launch_sub<2>(p, d_coef, dR, dS, dD, d);
    return launch_sub<1>(p, d_coef, dR, dS, dD, d);
}

}  // namespace sfft
