// Step a4' : the correlation terms whose second factor is a basis function rather than an image.
//   Lambda_{tb,s}(alpha,beta) = sum_{x,y} R^tb(x,y) T'_s((x+alpha) mod H, (y+beta) mod W)        (B8)
//   Delta_s                   = sum_{x,y} S(x,y) T'_s(x,y)                                        (B16, DESIGN g2)
// With T_tb = f_ib(x) g_jb(y) and T'_s = f'_i(x) g'_j(y) both are separable, so instead of the paper's
// full-size DFT products they are two small real dense contractions (FP64 tensor cores):
//   Q [x][(jb,j,beta)]  = sum_y R(x,y) * cy[(jb,j,beta)][y],     cy = g_jb(y) g'_j((y+beta) mod W)   (plan constant)
//   C [(ib,i,alpha)][(jb,j,beta)] = sum_x fx[(ib,i,alpha)][x] * Q[x][(jb,j,beta)],  fx = f_ib(x) f'_i((x+alpha) mod H)
//   Lambda_{(ib,jb),(i,j)}(alpha,beta) = C[(ib,i,alpha)][(jb,j,beta)]
//   QS[x][j] = sum_y S(x,y) g'_j(y),   Delta_(i,j) = sum_x f'_i(x) QS[x][j]
// Phi(0,0) = M_bb does not depend on the images and is a plan constant (plan.cu).
//
// k_dgemm : generic C = alpha A B(^T) + beta C, 64x64 CTA tile, mma.sync.m8n8k4.f64; also used by solve.cu.
#include <algorithm>

#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int BM = 64, BN = 64, BK = 16, LDS_ = BK + 4;   // smem row stride = 4 mod 16 doubles: conflict-free fragments

// grid: x = N tile, y = M tile, z = problem * ksplit + kpart.  block: 128 (2x2 warps of 32x32).
template <bool BT>
__global__ void __launch_bounds__(128) k_dgemm(GemmArgs g) {
    __shared__ double As[BM][LDS_];
    __shared__ double Bs[BN][LDS_];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int zi = blockIdx.z / g.ksplit, kp = blockIdx.z - zi * g.ksplit;
    const int i0 = blockIdx.y * BM, j0 = blockIdx.x * BN;
    if (g.lower && j0 > i0 + BM - 1) return;
    const double *A = g.A + (size_t)zi * g.sA, *B = g.B + (size_t)zi * g.sB;
    double *C = g.C + (size_t)zi * g.sC + (size_t)kp * g.sCk;
    const int klen = (g.K + g.ksplit - 1) / g.ksplit, kbeg = kp * klen, kend = min(g.K, kbeg + klen);
    const int wm = (warp >> 1) * 32, wn = (warp & 1) * 32, r = lane >> 2, kq = lane & 3;

    double acc[4][4][2];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

    // global -> register prefetch of the next K tile overlaps the MMAs of the current one
    double ra[BM * BK / 128], rb[BN * BK / 128];
    auto fetch = [&](int k0) {
        const int ka0 = g.kmodA > 0 ? k0 % g.kmodA : k0;
#pragma unroll
        for (int q = 0; q < BM * BK / 128; ++q) {
            const int i = tid + 128 * q, rr = i >> 4, kk = i & 15;
            ra[q] = (i0 + rr < g.M && k0 + kk < kend) ? __ldg(&A[(size_t)(i0 + rr) * g.lda + ka0 + kk]) : 0.0;
        }
        if (BT) {
#pragma unroll
            for (int q = 0; q < BN * BK / 128; ++q) {
                const int i = tid + 128 * q, rr = i >> 4, kk = i & 15;
                rb[q] = (j0 + rr < g.N && k0 + kk < kend) ? __ldg(&B[(size_t)(j0 + rr) * g.ldb + k0 + kk]) : 0.0;
            }
        } else {
#pragma unroll
            for (int q = 0; q < BN * BK / 128; ++q) {
                const int i = tid + 128 * q, kk = i >> 6, nn = i & 63;
                rb[q] = (j0 + nn < g.N && k0 + kk < kend) ? __ldg(&B[(size_t)(k0 + kk) * g.ldb + j0 + nn]) : 0.0;
            }
        }
    };
    if (kbeg < kend) fetch(kbeg);
    for (int k0 = kbeg; k0 < kend; k0 += BK) {
        __syncthreads();
#pragma unroll
        for (int q = 0; q < BM * BK / 128; ++q) {
            const int i = tid + 128 * q;
            As[i >> 4][i & 15] = ra[q];
        }
#pragma unroll
        for (int q = 0; q < BN * BK / 128; ++q) {
            const int i = tid + 128 * q;
            if (BT) Bs[i >> 4][i & 15] = rb[q];
            else Bs[i & 63][i >> 6] = rb[q];
        }
        __syncthreads();
        if (k0 + BK < kend) fetch(k0 + BK);
#pragma unroll
        for (int ks = 0; ks < BK; ks += 4) {
            double af[4], bf[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) af[a] = As[wm + 8 * a + r][ks + kq];
#pragma unroll
            for (int b = 0; b < 4; ++b) bf[b] = Bs[wn + 8 * b + r][ks + kq];
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) dmma884(acc[a][b], af[a], bf[b]);
        }
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b)
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int i = i0 + wm + 8 * a + r, j = j0 + wn + 8 * b + 2 * kq + q;
                if (i < g.M && j < g.N && (!g.lower || j <= i)) {
                    double *c = &C[(size_t)i * g.ldc + j];
                    *c = (g.beta == 0.0) ? g.alpha * acc[a][b][q] : fma(g.alpha, acc[a][b][q], g.beta * *c);
                }
            }
}

// Lambda table  la[((tb*FB + s)*L + ai)*L + bi] = sum_kpart C[kpart][(ib,i,ai)][(jb,j,bi)]
__global__ void k_lambda_pick(const double *__restrict__ C, double *__restrict__ tab, const int *__restrict__ kti,
                              const int *__restrict__ ktj, const int *__restrict__ bti, const int *__restrict__ btj, int FK,
                              int FB, int L, int nBa, int NC, int ksplit, size_t off_la, size_t tab_size) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, bz = blockIdx.y, LL = L * L;
    if (i >= FK * FB * LL) return;
    const int bi = i % L, ai = (i / L) % L, s = (i / LL) % FB, tb = i / (LL * FB);
    const int rowc = (kti[tb] * nBa + bti[s]) * L + ai, colc = (ktj[tb] * nBa + btj[s]) * L + bi;
    const double *c = C + (size_t)bz * ksplit * NC * NC + (size_t)rowc * NC + colc;
    double v = 0.0;
    for (int q = 0; q < ksplit; ++q) v += c[(size_t)q * NC * NC];
    tab[(size_t)bz * tab_size + off_la + i] = v;
}

// QS[x][j] = sum_y S(x,y) g'_j(y): one warp per image row, S streamed once (HBM-bound), NJ >= nBa accumulators per lane
template <int NJ>
__global__ void __launch_bounds__(256) k_rowdot(const double *__restrict__ S, const double *__restrict__ gB,
                                                double *__restrict__ QS, int H, int W, int nBa) {
    const int lane = threadIdx.x & 31, x = blockIdx.x * 8 + (threadIdx.x >> 5), bz = blockIdx.y;
    if (x >= H) return;
    const double2 *src = reinterpret_cast<const double2 *>(S + ((size_t)bz * H + x) * W);
    double acc[NJ];
#pragma unroll
    for (int j = 0; j < NJ; ++j) acc[j] = 0.0;
    for (int y2 = lane; y2 < W / 2; y2 += 32) {
        const double2 v = __ldg(&src[y2]);
#pragma unroll
        for (int j = 0; j < NJ; ++j)
            if (j < nBa) {
                const double2 gg = __ldg(reinterpret_cast<const double2 *>(gB + (size_t)j * W) + y2);
                acc[j] = fma(v.x, gg.x, fma(v.y, gg.y, acc[j]));
            }
    }
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
        double v = acc[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0 && j < nBa) QS[((size_t)bz * H + x) * nBa + j] = v;
    }
}

// POLY: row power moments  out[x][a] = sum_y img(x,y) u_y^a,  u_y = (2y+1)/W - 1  (exact in double), a < na.
// One warp per image row, four independent 16-byte loads in flight per lane; grid.y selects the image
// (0: R -> mu with naR moments, 1: S -> QS with naS, since g'_j = u^j for the polynomial background).
template <int NA>
__global__ void __launch_bounds__(256) k_rowmom(const double *__restrict__ R, const double *__restrict__ S,
                                                double *__restrict__ mu, double *__restrict__ QS, int H, int W, int naR,
                                                int naS) {
    const int lane = threadIdx.x & 31, x = blockIdx.x * 8 + (threadIdx.x >> 5), bz = blockIdx.z;
    if (x >= H) return;
    const bool isS = blockIdx.y == 1;
    const int na = isS ? naS : naR;
    const double2 *src = reinterpret_cast<const double2 *>((isS ? S : R) + ((size_t)bz * H + x) * W);
    const double invW = 1.0 / W;
    double acc[NA];
#pragma unroll
    for (int a = 0; a < NA; ++a) acc[a] = 0.0;
    for (int y2 = lane; y2 < W / 2; y2 += 128) {
        double2 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) v[q] = (y2 + 32 * q < W / 2) ? __ldg(&src[y2 + 32 * q]) : make_double2(0.0, 0.0);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double u0 = (double)(4 * (y2 + 32 * q) + 1) * invW - 1.0, u1 = u0 + 2.0 * invW;
            double p0 = v[q].x, p1 = v[q].y;
#pragma unroll
            for (int a = 0; a < NA; ++a)
                if (a < na) { acc[a] += p0 + p1; p0 *= u0; p1 *= u1; }
        }
    }
    double *dst = isS ? QS + ((size_t)bz * H + x) * naS : mu + ((size_t)bz * H + x) * naR;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        double t = acc[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0 && a < na) dst[a] = t;
    }
}

// POLY: Q[x][c] from the row power moments mu[x][a] and the |beta| row pixels whose shifted partner wraps
// (tables cq, cwr of plan.cu).  One thread per (x, c).
__global__ void k_q_poly(const double *__restrict__ R, const double *__restrict__ mu, const double *__restrict__ cq,
                         const double *__restrict__ cwr, double *__restrict__ Q, int H, int W, int NC, int A, int L) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, bz = blockIdx.y;
    if (i >= H * NC) return;
    const int x = i / NC, c = i - x * NC, w = (L - 1) / 2, beta = c % L - w;
    const double *m = mu + ((size_t)bz * H + x) * A, *q = cq + (size_t)c * A;
    double v = 0.0;
    for (int a = 0; a < A; ++a) v = fma(__ldg(&q[a]), m[a], v);
    const double *row = R + ((size_t)bz * H + x) * W + (beta > 0 ? W - beta : 0);
    const int nb = beta > 0 ? beta : -beta;
    for (int k = 0; k < nb; ++k) v = fma(__ldg(&cwr[(size_t)c * w + k]), __ldg(&row[k]), v);
    Q[(size_t)bz * H * NC + i] = v;
}

// Delta_s = sum_x f'_i(x) QS[x][j]   (one 256-thread CTA per s)
__global__ void __launch_bounds__(256) k_delta(const double *__restrict__ QS, const double *__restrict__ xwt,
                                               const int *__restrict__ bti, const int *__restrict__ btj,
                                               double *__restrict__ tab, int H, int nKa, int nBa, int FB, size_t off_de,
                                               size_t tab_size) {
    const int s = blockIdx.x, bz = blockIdx.y, tid = threadIdx.x, lane = tid & 31;
    __shared__ double red[8];
    const double *f = xwt + (size_t)(nKa + bti[s]) * H;
    const double *q = QS + (size_t)bz * H * nBa + btj[s];
    double v = 0.0;
    for (int x = tid; x < H; x += 256) v = fma(f[x], q[(size_t)x * nBa], v);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) red[tid >> 5] = v;
    __syncthreads();
    if (tid == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; ++k) t += red[k];
        tab[(size_t)bz * tab_size + off_de + s] = t;
    }
}

}  // namespace

cudaError_t launch_dgemm(sfft_plan *p, const GemmArgs &g) {
    dim3 grid((g.N + BN - 1) / BN, (g.M + BM - 1) / BM, g.nz * g.ksplit);
    if (g.bT) k_dgemm<true><<<grid, 128, 0, p->stream>>>(g);
    else k_dgemm<false><<<grid, 128, 0, p->stream>>>(g);
    p->launches++;
    return cudaGetLastError();
}

cudaError_t launch_moments(sfft_plan *p, const double *dR, const double *dS) {
    const int H = p->H, W = p->W, NC = p->NC;
    const long long P = (long long)H * W;
    auto rowdot = [&](const double *img, const double *tabl, double *out, int nj) {
        dim3 grid((H + 7) / 8, p->nbatch);
        if (nj <= 4) k_rowdot<4><<<grid, 256, 0, p->stream>>>(img, tabl, out, H, W, nj);
        else if (nj <= 8) k_rowdot<8><<<grid, 256, 0, p->stream>>>(img, tabl, out, H, W, nj);
        else if (nj <= 12) k_rowdot<12><<<grid, 256, 0, p->stream>>>(img, tabl, out, H, W, nj);
        else k_rowdot<17><<<grid, 256, 0, p->stream>>>(img, tabl, out, H, W, nj);
        p->launches++;
    };
    cudaError_t e = cudaSuccess;
    if (p->basis == SFFT_BASIS_POLY) {
        // Q from nMom row power moments (one streaming pass over R) instead of the NC-column contraction
        const int na = std::max(p->nMom, p->nBa);
        dim3 grid((H + 7) / 8, 2, p->nbatch);
        if (na <= 3) k_rowmom<3><<<grid, 256, 0, p->stream>>>(dR, dS, p->mu, p->QS, H, W, p->nMom, p->nBa);
        else if (na <= 5) k_rowmom<5><<<grid, 256, 0, p->stream>>>(dR, dS, p->mu, p->QS, H, W, p->nMom, p->nBa);
        else if (na <= 9) k_rowmom<9><<<grid, 256, 0, p->stream>>>(dR, dS, p->mu, p->QS, H, W, p->nMom, p->nBa);
        else k_rowmom<17><<<grid, 256, 0, p->stream>>>(dR, dS, p->mu, p->QS, H, W, p->nMom, p->nBa);
        p->launches++;
        k_q_poly<<<dim3((H * NC + 255) / 256, p->nbatch), 256, 0, p->stream>>>(dR, p->mu, p->dt.cq, p->dt.cwr, p->Q, H, W, NC,
                                                                           p->nMom, p->L);
        p->launches++;
    } else {
    // Q = R * cy^T
    GemmArgs g{};
    g.A = dR; g.B = p->dt.cy; g.C = p->Q; g.M = H; g.N = NC; g.K = W; g.lda = W; g.ldb = W; g.ldc = NC;
    g.sA = P; g.sB = 0; g.sC = (long long)p->ksq * H * NC; g.sCk = (long long)H * NC; g.nz = p->nbatch; g.ksplit = p->ksq;
    g.alpha = 1.0; g.beta = 0.0; g.bT = true; g.lower = false; g.kmodA = 0;
    e = launch_dgemm(p, g);
    if (e != cudaSuccess) return e;
    }
    // QS = S * gB^T  (POLY: done by k_rowmom above)
    if (p->basis != SFFT_BASIS_POLY) rowdot(dS, p->dt.gB, p->QS, p->nBa);
    // C = fx * (sum of the ksq partial Q's): K = ksq stacked copies of the x axis, split in ksq*ksplit parts
    const int parts = p->ksq * p->ksplit;
    GemmArgs h{};
    h.A = p->dt.fx; h.B = p->Q; h.C = p->LamC; h.M = NC; h.N = NC; h.K = p->ksq * H; h.lda = H; h.ldb = NC; h.ldc = NC;
    h.sA = 0; h.sB = (long long)p->ksq * H * NC; h.sC = (long long)parts * NC * NC; h.sCk = (long long)NC * NC;
    h.nz = p->nbatch; h.ksplit = parts; h.alpha = 1.0; h.beta = 0.0; h.bT = false; h.lower = false; h.kmodA = H;
    e = launch_dgemm(p, h);
    if (e != cudaSuccess) return e;
    const int tot = p->FK * p->FB * p->L * p->L;
    k_lambda_pick<<<dim3((tot + 255) / 256, p->nbatch), 256, 0, p->stream>>>(
        p->LamC, p->tab, p->dt.kti, p->dt.ktj, p->dt.bti, p->dt.btj, p->FK, p->FB, p->L, p->nBa, NC, parts, p->off_la,
        p->tab_size);
    k_delta<<<dim3(p->FB, p->nbatch), 256, 0, p->stream>>>(p->QS, p->dt.xwt, p->dt.bti, p->dt.btj, p->tab, H, p->nKa, p->nBa,
                                                         p->FB, p->off_de, p->tab_size);
    p->launches += 2;
    return cudaGetLastError();
}

}  // namespace sfft
