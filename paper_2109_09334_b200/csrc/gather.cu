// Step a5: the lag gather.  Every entry of the normal matrix of Eq. 18 is a
// sum/difference of at most four values of the lag tables (App. B):
//   (B5, reading DESIGN g1)  both lags != 0 : Om(ab-a) - Om(ab) - Om(-a) + Om(0)
//                            only a  = 0    : Om(ab) - Om(0)
//                            only ab = 0    : Om(-a) - Om(0)
//                            both 0         : Om(0)
//   (B7/B9)  M_ab = La(ab) - La(0) | La(0);   (B11) M_bb = Phi(0,0) (plan constant)
//   (B13)    rhs_a = Th(ab) - Th(0) | Th(0);  (B15) rhs_b = De(0,0)
// with Om_{tb,t}(rho) = Om_{t,tb}(-rho) for tb > t.  Real-space scaling: M = Phi^T Phi.
// One warp fills a 32-entry run of a matrix row, so stores are 256-byte coalesced; both
// triangles are written from the (min,max)-ordered index pair, which makes M exactly symmetric.
#include <algorithm>

#include "sfft_internal.h"

namespace sfft {
namespace {

struct GatherDims { int FK, FB, L, w, n, nO, LL, ns, cpr, nshare, rshare; size_t off_om, off_th, off_la, off_de, tab_size; };

__device__ __forceinline__ double omega(const double *om, const GatherDims &d, int tb, int t, int rho, int eps) {
    if (tb > t) { int q = tb; tb = t; t = q; rho = -rho; eps = -eps; }
    int pair = tb * d.FK - tb * (tb - 1) / 2 + (t - tb);
    return om[((size_t)pair * d.nO + (rho + d.L - 1)) * d.nO + (eps + d.L - 1)];
}

// entry (kb <= k) of the full normal matrix, from the lag tables
// kdec[k] = t << 16 | (alpha + w) << 8 | (beta + w) for a kernel unknown k (plan table: no integer divisions here)
__device__ __forceinline__ double m_entry(const double *om, const double *la, const double *phi0, const int *kdec,
                                          const GatherDims &d, int kb, int k) {
    const int na = d.FK * d.LL;
    if (k < na) {
        const int db = __ldg(&kdec[kb]), dk = __ldg(&kdec[k]);
        const int tbar = db >> 16, t = dk >> 16;
        const int alb = ((db >> 8) & 255) - d.w, beb = (db & 255) - d.w, al = ((dk >> 8) & 255) - d.w, be = (dk & 255) - d.w;
        bool cb = (alb == 0 && beb == 0), c = (al == 0 && be == 0);
        double o0 = omega(om, d, tbar, t, 0, 0);
        if (cb && c) return o0;
        if (c) return omega(om, d, tbar, t, alb, beb) - o0;
        if (cb) return omega(om, d, tbar, t, -al, -be) - o0;
        return (omega(om, d, tbar, t, alb - al, beb - be) - omega(om, d, tbar, t, alb, beb)) -
               (omega(om, d, tbar, t, -al, -be) - o0);
    }
    if (kb < na) {
        const int db = __ldg(&kdec[kb]);
        const int tbar = db >> 16, ab = ((db >> 8) & 255) * d.L + (db & 255), s = k - na;
        const double *l = la + ((size_t)tbar * d.FB + s) * d.LL;
        double l0 = l[d.w * d.L + d.w];
        return (ab == d.w * d.L + d.w) ? l0 : l[ab] - l0;
    }
    return phi0[(size_t)(kb - na) * d.FB + (k - na)];
}

__device__ __forceinline__ double rhs_entry(const double *th, const double *de, const GatherDims &d, int k) {
    const int na = d.FK * d.LL;
    if (k >= na) return de[k - na];
    int tbar = k / d.LL, ab = k % d.LL;
    const double *t0 = th + (size_t)tbar * d.LL;
    double c0 = t0[d.w * d.L + d.w];
    return (ab == d.w * d.L + d.w) ? c0 : t0[ab] - c0;
}

// Reduced systems (constant photometric ratio; rectangular kernels): solved unknown r
// stands for the full-layout unknown ridx[r] (plan table).  Under the constant photometric ratio the shared unknown
// at r = rshare stands for `nshare` centre entries t*LL + a0, t < nshare (1: POLY, the others are zero; F_K:
// BSPLINE, all equal).  M' = C^T M C is formed entry by entry.
__global__ void k_gather(const double *__restrict__ tab, const double *__restrict__ phi0, const int *__restrict__ kdec,
                         const int *__restrict__ ridx, double *__restrict__ M, double *__restrict__ rhs, GatherDims d) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y, b = blockIdx.z;
    if (col >= d.ns) return;
    const double *tb_ = tab + (size_t)b * d.tab_size;
    const double *om = tb_ + d.off_om, *th = tb_ + d.off_th, *la = tb_ + d.off_la, *de = tb_ + d.off_de;
    // ordered pair (lo <= hi) so that M[row][col] and M[col][row] run the same arithmetic
    const int lo = min(row, col), hi = max(row, col);
    const int klo = __ldg(&ridx[lo]), khi = __ldg(&ridx[hi]);
    const int nlo = (lo == d.rshare) ? d.nshare : 1, nhi = (hi == d.rshare) ? d.nshare : 1;
    double v = 0.0;
    for (int p = 0; p < nlo; ++p)
        for (int q = 0; q < nhi; ++q) {
            const int k1 = klo + p * d.LL, k2 = khi + q * d.LL;
            v += m_entry(om, la, phi0, kdec, d, min(k1, k2), max(k1, k2));
        }
    M[((size_t)b * d.ns + row) * d.ns + col] = v;
    if (row == 0) {   // the first row of CTAs also fills the right-hand side
        const int kc = __ldg(&ridx[col]), nc = (col == d.rshare) ? d.nshare : 1;
        double r = 0.0;
        for (int q = 0; q < nc; ++q) r += rhs_entry(th, de, d, kc + q * d.LL);
        rhs[(size_t)b * d.ns + col] = r;
    }
}

// Kernel-kernel part of M for the unconstrained system: CTA (t-group, tb, chunk) fills kGatherRows rows of the blocks
// M[(tb, .)][(t, .)], t in the group, from the Omega tables of the pairs (min, max)(tb, t) staged in shared memory (one
// table read per CTA instead of four L2 reads per entry).  A warp writes its row across ALL blocks of the group, i.e.
// one contiguous run of TG L^2 entries: the block boundaries (L^2 entries = a fraction of a 32-byte sector) are then
// written by the same warp back to back instead of by different CTAs at different times, which is what made the
// 31 GB write of config 5 run at 16 % of the HBM roofline.  Entries are formed from the (lower, higher)-ordered
// unknown pair exactly as in m_entry, so M stays exactly symmetric.
constexpr int kGatherRows = 32;
__global__ void __launch_bounds__(256) k_gather_kk(const double *__restrict__ tab, double *__restrict__ M, GatherDims d,
                                                   int nchunk, int TG) {
    extern __shared__ double som[];                       // [TG][nO][nO] Omega of the ordered pairs, then int dec[LL]
    const int nO2 = d.nO * d.nO;
    int *dec = reinterpret_cast<int *>(som + (size_t)TG * nO2);
    const int t0 = blockIdx.x * TG, tg = min(TG, d.FK - t0), tb = blockIdx.y, b = blockIdx.z / nchunk,
              chunk = blockIdx.z - b * nchunk;
    for (int i = threadIdx.x; i < tg * nO2; i += 256) {
        const int tl = i / nO2, t = t0 + tl, tlo = min(tb, t), thi = max(tb, t);
        const int pair = tlo * d.FK - tlo * (tlo - 1) / 2 + (thi - tlo);
        som[i] = __ldg(&tab[(size_t)b * d.tab_size + d.off_om + (size_t)pair * nO2 + (i - tl * nO2)]);
    }
    for (int a = threadIdx.x; a < d.LL; a += 256) dec[a] = ((a / d.L - d.w) << 16) | ((a % d.L - d.w) & 0xffff);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, c0 = (d.L - 1) * d.nO + (d.L - 1);   // index of lag (0,0)
    const int r1 = min(d.LL, (chunk + 1) * kGatherRows);
    for (int ab = chunk * kGatherRows + warp; ab < r1; ab += 8) {
        const int kb = tb * d.LL + ab, dab = dec[ab];
        double *row = M + ((size_t)b * d.ns + kb) * d.ns + (size_t)t0 * d.LL;
        for (int tl = 0; tl < tg; ++tl) {
            const double *so = som + (size_t)tl * nO2;
            const double o0 = so[c0];
            const int t = t0 + tl;
            for (int a = lane; a < d.LL; a += 32) {
                const int k = t * d.LL + a;
                // (first, second) = the unknowns in increasing index order
                const int df = kb <= k ? dab : dec[a], ds = kb <= k ? dec[a] : dab;
                const int alb = df >> 16, beb = (short)(df & 0xffff), al = ds >> 16, be = (short)(ds & 0xffff);
                const bool cb = (alb == 0 && beb == 0), c = (al == 0 && be == 0);
                double v;
                if (cb && c) v = o0;
                else if (c) v = so[c0 + alb * d.nO + beb] - o0;
                else if (cb) v = so[c0 - al * d.nO - be] - o0;
                else v = (so[c0 + (alb - al) * d.nO + (beb - be)] - so[c0 + alb * d.nO + beb]) - (so[c0 - al * d.nO - be] - o0);
                row[tl * d.LL + a] = v;
            }
        }
    }
}

// Background part of the unconstrained system: columns and rows of the F_B background unknowns (B7/B9, B11), and the
// right-hand side (B13, B15).  thread = unknown i, blockIdx.y = background term s; both M[i][na+s] and M[na+s][i].
__global__ void __launch_bounds__(128) k_gather_bg(const double *__restrict__ tab, const double *__restrict__ phi0,
                                                   const int *__restrict__ kdec, double *__restrict__ M,
                                                   double *__restrict__ rhs, GatherDims d) {
    const int i = blockIdx.x * 128 + threadIdx.x, s = blockIdx.y, b = blockIdx.z;
    if (i >= d.n) return;
    const double *tb_ = tab + (size_t)b * d.tab_size;
    const double *om = tb_ + d.off_om, *th = tb_ + d.off_th, *la = tb_ + d.off_la, *de = tb_ + d.off_de;
    const int k = d.FK * d.LL + s;
    const double v = m_entry(om, la, phi0, kdec, d, min(i, k), max(i, k));
    M[((size_t)b * d.ns + i) * d.ns + k] = v;
    M[((size_t)b * d.ns + k) * d.ns + i] = v;
    if (s == 0) rhs[(size_t)b * d.ns + i] = rhs_entry(th, de, d, i);
}

// c = C c': reduced solution -> full coefficient layout (fmap[k] = solved index of full unknown k, -1 = zero)
__global__ void k_expand_coef(const double *__restrict__ cr, double *__restrict__ c, const int *__restrict__ fmap, int n,
                              int ns) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (k >= n) return;
    const int r = __ldg(&fmap[k]);
    c[(size_t)b * n + k] = r >= 0 ? cr[(size_t)b * ns + r] : 0.0;
}

}  // namespace

static GatherDims gather_dims(const sfft_plan *p) {
    return GatherDims{p->FK, p->FB, p->L, p->w, p->n, 2 * p->L - 1, p->L * p->L, p->ns, p->cpr,
                      p->basis == SFFT_BASIS_POLY ? 1 : p->FK, p->cpr ? p->rshare : -1, p->off_om, p->off_th, p->off_la, p->off_de, p->tab_size};
}

cudaError_t launch_gather(sfft_plan *p) {
    GatherDims d = gather_dims(p);
    if (!p->reduced) {
        const int nchunk = (d.LL + kGatherRows - 1) / kGatherRows;
        // blocks per CTA: as many Omega tables as fit ~96 KB, at most 16, and enough CTAs left to fill the machine
        int TG = std::max(1, std::min(16, (int)((96 * 1024) / ((size_t)d.nO * d.nO * sizeof(double)))));
        TG = std::min(TG, p->FK);
        while (TG > 1 && (long)((p->FK + TG - 1) / TG) * p->FK * p->nbatch * nchunk < 2 * 148) TG = (TG + 1) / 2;
        const size_t smem = (size_t)TG * d.nO * d.nO * sizeof(double) + (size_t)d.LL * sizeof(int);
        cudaError_t e = cudaFuncSetAttribute(k_gather_kk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k_gather_kk<<<dim3((p->FK + TG - 1) / TG, p->FK, p->nbatch * nchunk), 256, smem, p->stream>>>(p->tab, p->M, d, nchunk, TG);
        k_gather_bg<<<dim3((p->n + 127) / 128, p->FB, p->nbatch), 128, 0, p->stream>>>(p->tab, p->dt.phi0, p->dt.kdec, p->M,
                                                                                     p->rhs, d);
        p->launches += 2;
        return cudaGetLastError();
    }
    dim3 grid((p->ns + 127) / 128, p->ns, p->nbatch);
    k_gather<<<grid, 128, 0, p->stream>>>(p->tab, p->dt.phi0, p->dt.kdec, p->dt.ridx, p->M, p->rhs, d);
    p->launches++;
    return cudaGetLastError();
}

cudaError_t launch_expand_coef(sfft_plan *p, const double *d_cr, double *d_coef) {
    k_expand_coef<<<dim3((p->n + 255) / 256, p->nbatch), 256, 0, p->stream>>>(d_cr, d_coef, p->dt.fmap, p->n, p->ns);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
