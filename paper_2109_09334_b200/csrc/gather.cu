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

struct GatherDims { int FK, FB, L, w, n, nO, LL; size_t off_om, off_th, off_la, off_de, tab_size; };

__device__ __forceinline__ double omega(const double *om, const GatherDims &d, int tb, int t, int rho, int eps) {
    if (tb > t) { int q = tb; tb = t; t = q; rho = -rho; eps = -eps; }
    int pair = tb * d.FK - tb * (tb - 1) / 2 + (t - tb);
    return om[((size_t)pair * d.nO + (rho + d.L - 1)) * d.nO + (eps + d.L - 1)];
}

__global__ void k_gather(const double *__restrict__ tab, const double *__restrict__ phi0, double *__restrict__ M,
                         double *__restrict__ rhs, GatherDims d) {
    const int col = blockIdx.x * blockDim.x + threadIdx.x, row = blockIdx.y, b = blockIdx.z;
    if (col >= d.n) return;
    const double *tb_ = tab + (size_t)b * d.tab_size;
    const double *om = tb_ + d.off_om, *th = tb_ + d.off_th, *la = tb_ + d.off_la, *de = tb_ + d.off_de;
    const int na = d.FK * d.LL;
    // ordered pair (kb <= k) so that M[row][col] and M[col][row] run the same arithmetic
    const int kb = min(row, col), k = max(row, col);
    double v;
    if (k < na) {
        int tbar = kb / d.LL, ab = kb % d.LL, t = k / d.LL, a = k % d.LL;
        int alb = ab / d.L - d.w, beb = ab % d.L - d.w, al = a / d.L - d.w, be = a % d.L - d.w;
        bool cb = (alb == 0 && beb == 0), c = (al == 0 && be == 0);
        double o0 = omega(om, d, tbar, t, 0, 0);
        if (cb && c) v = o0;
        else if (c) v = omega(om, d, tbar, t, alb, beb) - o0;
        else if (cb) v = omega(om, d, tbar, t, -al, -be) - o0;
        else v = (omega(om, d, tbar, t, alb - al, beb - be) - omega(om, d, tbar, t, alb, beb)) -
                 (omega(om, d, tbar, t, -al, -be) - o0);
    } else if (kb < na) {
        int tbar = kb / d.LL, ab = kb % d.LL, s = k - na;
        const double *l = la + ((size_t)tbar * d.FB + s) * d.LL;
        double l0 = l[d.w * d.L + d.w];
        v = (ab == d.w * d.L + d.w) ? l0 : l[ab] - l0;
    } else {
        v = phi0[(size_t)(kb - na) * d.FB + (k - na)];
    }
    M[((size_t)b * d.n + row) * d.n + col] = v;
    if (row == 0) {   // the first row of CTAs also fills the right-hand side
        double r;
        if (col < na) {
            int tbar = col / d.LL, ab = col % d.LL;
            const double *t0 = th + (size_t)tbar * d.LL;
            double c0 = t0[d.w * d.L + d.w];
            r = (ab == d.w * d.L + d.w) ? c0 : t0[ab] - c0;
        } else {
            r = de[col - na];
        }
        rhs[(size_t)b * d.n + col] = r;
    }
}

}  // namespace

cudaError_t launch_gather(sfft_plan *p) {
    GatherDims d{p->FK, p->FB, p->L, p->w, p->n, 2 * p->L - 1, p->L * p->L,
                 p->off_om, p->off_th, p->off_la, p->off_de, p->tab_size};
    dim3 grid((p->n + 127) / 128, p->n, p->nbatch);
    k_gather<<<grid, 128, 0, p->stream>>>(p->tab, p->dt.phi0, p->M, p->rhs, d);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
