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
#include "sfft_internal.h"

namespace sfft {
namespace {

struct GatherDims { int FK, FB, L, w, n, nO, LL, ns, cpr, nshare; size_t off_om, off_th, off_la, off_de, tab_size; };

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

// Full index of reduced unknown r (constant photometric ratio: the centre coefficients of the
// terms t >= 1 are not free).  The shared unknown sits at r = a0; it stands for `nshare` centre entries
// t*LL + a0, t < nshare (1: POLY, the others are zero; F_K: BSPLINE, all equal).
__device__ __forceinline__ int full_index(const GatherDims &d, int r) {
    const int a0 = d.w * d.L + d.w;
    if (!d.cpr || r < d.LL) return r;
    const int na_r = d.FK * d.LL - (d.FK - 1);
    if (r >= na_r) return r + (d.FK - 1);
    const int q = r - d.LL, t = 1 + q / (d.LL - 1), a = q % (d.LL - 1);
    return t * d.LL + (a < a0 ? a : a + 1);
}

__global__ void k_gather(const double *__restrict__ tab, const double *__restrict__ phi0, const int *__restrict__ kdec,
                         double *__restrict__ M, double *__restrict__ rhs, GatherDims d) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y, b = blockIdx.z;
    if (col >= d.ns) return;
    const double *tb_ = tab + (size_t)b * d.tab_size;
    const double *om = tb_ + d.off_om, *th = tb_ + d.off_th, *la = tb_ + d.off_la, *de = tb_ + d.off_de;
    const int a0 = d.w * d.L + d.w;
    // ordered pair (lo <= hi) so that M[row][col] and M[col][row] run the same arithmetic
    const int lo = min(row, col), hi = max(row, col);
    const int klo = full_index(d, lo), khi = full_index(d, hi);
    const int nlo = (d.cpr && lo == a0) ? d.nshare : 1, nhi = (d.cpr && hi == a0) ? d.nshare : 1;
    double v = 0.0;
    for (int p = 0; p < nlo; ++p)
        for (int q = 0; q < nhi; ++q) {
            const int k1 = klo + p * d.LL, k2 = khi + q * d.LL;
            v += m_entry(om, la, phi0, kdec, d, min(k1, k2), max(k1, k2));
        }
    M[((size_t)b * d.ns + row) * d.ns + col] = v;
    if (row == 0) {   // the first row of CTAs also fills the right-hand side
        const int kc = full_index(d, col), nc = (d.cpr && col == a0) ? d.nshare : 1;
        double r = 0.0;
        for (int q = 0; q < nc; ++q) r += rhs_entry(th, de, d, kc + q * d.LL);
        rhs[(size_t)b * d.ns + col] = r;
    }
}

// c = C c': reduced solution -> full coefficient layout (constrained centre entries filled in)
__global__ void k_expand_coef(const double *__restrict__ cr, double *__restrict__ c, GatherDims d, int poly) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (k >= d.n) return;
    const int a0 = d.w * d.L + d.w, na = d.FK * d.LL;
    double v;
    if (k < na && k % d.LL == a0) {
        v = (k / d.LL == 0 || !poly) ? cr[(size_t)b * d.ns + a0] : 0.0;
    } else if (k < na) {
        const int t = k / d.LL, a = k % d.LL;
        const int r = t == 0 ? a : d.LL + (t - 1) * (d.LL - 1) + (a < a0 ? a : a - 1);
        v = cr[(size_t)b * d.ns + r];
    } else {
        v = cr[(size_t)b * d.ns + (k - (d.FK - 1))];
    }
    c[(size_t)b * d.n + k] = v;
}

}  // namespace

static GatherDims gather_dims(const sfft_plan *p) {
    return GatherDims{p->FK, p->FB, p->L, p->w, p->n, 2 * p->L - 1, p->L * p->L, p->ns, p->cpr,
                      p->basis == SFFT_BASIS_POLY ? 1 : p->FK, p->off_om, p->off_th, p->off_la, p->off_de, p->tab_size};
}

cudaError_t launch_gather(sfft_plan *p) {
    GatherDims d = gather_dims(p);
    dim3 grid((p->ns + 127) / 128, p->ns, p->nbatch);
    k_gather<<<grid, 128, 0, p->stream>>>(p->tab, p->dt.phi0, p->dt.kdec, p->M, p->rhs, d);
    p->launches++;
    return cudaGetLastError();
}

cudaError_t launch_expand_coef(sfft_plan *p, const double *d_cr, double *d_coef) {
    GatherDims d = gather_dims(p);
    k_expand_coef<<<dim3((p->n + 255) / 256, p->nbatch), 256, 0, p->stream>>>(d_cr, d_coef, d, p->basis == SFFT_BASIS_POLY);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
