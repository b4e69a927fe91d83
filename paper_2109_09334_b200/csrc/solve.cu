// Step a6: dense FP64 solve of the SPD normal system (DESIGN g11).
//
//   1. Jacobi scaling  A = D M D, D = diag(M)^-1/2  (removes the 10^6..10^12 spread between
//      kernel and background unknowns), rhs appended as an extra ROW of the lower triangle:
//      factoring [[A, .],[r^T D, .]] leaves z = L^-1 D r in that row, so the forward
//      substitution comes for free with the panel solves.
//   2. Right-looking blocked Cholesky with one look-ahead step, panel width NB = 64, ONE launch
//      per panel (k_chol_step).  Launch k holds three kinds of CTA:
//        P  (one per 64-row slab below the diagonal block of panel k): applies panel k-1 to its
//           rows of column strip k and to the diagonal block (FP64 tensor cores), factors the
//           64x64 diagonal block (every P CTA redundantly - that is cheaper than another launch),
//           and solves its slab against it;
//        U  (one per 64x64 tile of the lower triangle right of strip k): rank-64 update with
//           panel k-1 on the FP64 tensor cores (mma.sync.m8n8k4.f64: a dense contraction);
//        I  (one): inverse of the diagonal block of panel k-1, used by the back substitution.
//      P(k) needs only panel k-1 and the U updates of launch k-1, so the latency-bound panel
//      chain (factor + triangular solve) overlaps the throughput-bound trailing update.
//   3. Backward substitution L^T y = z by a thread-block cluster of 8 CTAs per system: the owner
//      of diagonal block b forms y_b = W_b^T z_b (W_b = L_bb^-1 from the I CTAs), broadcasts it
//      through distributed shared memory, and every CTA updates the columns it owns.  c = D y.
// A non-positive pivot writes its index to flag[2*b] (reported as SFFT_ERR_NOT_SPD).
#include <cooperative_groups.h>

#include <algorithm>

#include "sfft_internal.h"

namespace cg = cooperative_groups;

namespace sfft {
namespace {

constexpr int NB = 64;        // panel width = tile size
constexpr int LDT = NB + 4;   // smem stride of MMA operand tiles (= 4 mod 16: conflict-free fragments)
constexpr int LDX = NB + 1;   // smem stride of the factor / solve views (conflict-free row-per-thread access)
constexpr int CS = 8;         // cluster size of the back substitution

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}

__global__ void k_scale_diag(const double *__restrict__ M, double *__restrict__ dscale, int *flag, int n) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (i >= n) return;
    double d = M[((size_t)b * n + i) * n + i];
    if (!(d > 0.0)) { atomicCAS(&flag[2 * b], -1, i); d = 1.0; }
    dscale[(size_t)b * n + i] = rsqrt(d);
}

// Lf[i][j] = M[i][j] d_i d_j (j <= i), row n = rhs_j d_j
__global__ void k_scale_copy(const double *__restrict__ M, const double *__restrict__ rhs,
                             const double *__restrict__ dscale, double *__restrict__ Lf, int n, int ldl) {
    int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y, b = blockIdx.z;
    if (j >= n || j > i) return;
    const double *d = dscale + (size_t)b * n;
    double v = (i < n) ? M[((size_t)b * n + i) * n + j] * d[i] * d[j] : rhs[(size_t)b * n + j] * d[j];
    Lf[((size_t)b * (n + 1) + i) * ldl + j] = v;
}

// T[r][c] = L[row0 + r][col0 + c] for r < nr (else 0), 64 columns, into an MMA operand tile (stride LDT)
__device__ __forceinline__ void load_tile(double *T, const double *__restrict__ L, int ldl, int row0, int col0, int nr) {
    for (int i = threadIdx.x; i < NB * NB / 2; i += 256) {
        const int r = i >> 5, c = (i & 31) * 2;
        double2 v = make_double2(0.0, 0.0);
        if (r < nr) v = *reinterpret_cast<const double2 *>(&L[(size_t)(row0 + r) * ldl + col0 + c]);
        T[r * LDT + c] = v.x;
        T[r * LDT + c + 1] = v.y;
    }
}

// acc += A B^T for 64x64x64 operand tiles in shared memory; warp w owns rows 16*(w>>1).., cols 32*(w&1)..
// acc[a][b][q] <-> row 16*(w>>1) + 8a + (lane>>2), col 32*(w&1) + 8b + 2*(lane&3) + q
__device__ __forceinline__ void mma_64(const double *A, const double *B, double (&acc)[2][4][2]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, r = lane >> 2, kq = lane & 3;
    const double *ap = A + ((warp >> 1) * 16 + r) * LDT + kq;
    const double *bp = B + ((warp & 1) * 32 + r) * LDT + kq;
#pragma unroll 4
    for (int k = 0; k < NB; k += 4) {
        double af[2], bf[4];
#pragma unroll
        for (int a = 0; a < 2; ++a) af[a] = ap[a * 8 * LDT + k];
#pragma unroll
        for (int b = 0; b < 4; ++b) bf[b] = bp[b * 8 * LDT + k];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) dmma884(acc[a][b], af[a], bf[b]);
    }
}

// x L^T = a for one row held in registers (right-looking: after x[k] is final, the remaining
// entries receive its contribution, so the dependent chain is one FMA + one multiply per column).
// Ls = lower-triangular factor in shared memory (stride LDX), rs[k] = 1 / L[k][k].
__device__ __forceinline__ void row_trsm(double (&x)[NB], const double *Ls, const double *rs) {
#pragma unroll
    for (int k = 0; k < NB; ++k) {
        x[k] *= rs[k];
#pragma unroll
        for (int m = k + 1; m < NB; ++m) x[m] = fma(-x[k], Ls[m * LDX + k], x[m]);
    }
}

// In-place Cholesky of the 64x64 block Dg (shared memory, stride LDX, lower triangle valid, identity
// padded beyond nb) by all 256 threads.  Every thread keeps a 4x4 register tile (rows ty+16a, cols
// tx+16b); step k publishes column k through a double-buffered shared column, so there is ONE barrier
// per column; the column scaling by 1/sqrt(pivot) is deferred to the end.  rs[k] = 1/L[k][k] on exit.
__device__ __forceinline__ void chol_64(double *Dg, double *colbuf, double *pivs, double *rs, int nb, int *flag,
                                        int gidx0, bool report) {
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    double t[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) t[a][b] = Dg[(ty + 16 * a) * LDX + tx + 16 * b];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        for (int kk = 0; kk < 16; ++kk) {
            const int k = 16 * b + kk;
            if (k >= nb) break;                              // uniform
            double *cb = colbuf + (k & 1) * NB;
            if (tx == kk) {
#pragma unroll
                for (int a = 0; a < 4; ++a) cb[ty + 16 * a] = t[a][b];
            }
            __syncthreads();
            double piv = cb[k];
            if (!(piv > 0.0)) {
                if (report && tid == 0) atomicCAS(flag, -1, gidx0 + k);
                piv = 1.0;
            }
            if (tid == 0) pivs[k] = piv;
            const double inv = 1.0 / piv;
            double lr[4];
#pragma unroll
            for (int a = 0; a < 4; ++a) lr[a] = cb[ty + 16 * a];
#pragma unroll
            for (int bb = b; bb < 4; ++bb) {
                const double lc = cb[tx + 16 * bb] * inv;
                if (bb > b || tx > kk) {
#pragma unroll
                    for (int a = 0; a < 4; ++a) t[a][bb] = fma(-lr[a], lc, t[a][bb]);
                }
            }
        }
    }
    __syncthreads();
    if (tid < NB) rs[tid] = (tid < nb) ? rsqrt(pivs[tid]) : 1.0;
    __syncthreads();
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int r = ty + 16 * a, c = tx + 16 * b;
            double v = 0.0;
            if (c < r) v = (r < nb) ? t[a][b] * rs[c] : 0.0;
            else if (c == r) v = (r < nb) ? pivs[c] * rs[c] : 1.0;
            Dg[r * LDX + c] = v;
        }
    __syncthreads();
}

constexpr size_t kStepSmem = (size_t)(2 * NB * LDT + 2 * NB + NB + NB) * sizeof(double);

// One launch per panel k (see the header).  grid.x = nslab P CTAs, then ntiles U CTAs and one I CTA (k >= 1).
__global__ void __launch_bounds__(256) k_chol_step(double *__restrict__ Lf, double *__restrict__ Winv, int *flag, int n,
                                                   int ldl, int k, int nslab, int ntiles, int nblk) {
    extern __shared__ double sm[];
    double *T0 = sm, *T1 = sm + NB * LDT;                   // MMA operand tiles; later the factor / slab views
    double *colbuf = sm + 2 * NB * LDT, *pivs = colbuf + 2 * NB, *rs = pivs + NB;
    const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r8 = lane >> 2, kq = lane & 3, wm = (warp >> 1) * 16, wn = (warp & 1) * 32;
    double *L = Lf + (size_t)b * (n + 1) * ldl;
    const int j0 = k * NB, nb = min(NB, n - j0), j1 = j0 + nb, jp0 = j0 - NB;
    int bx = blockIdx.x;

    if (bx < nslab) {
        // ------------------------------ P: panel k ------------------------------
        const int r0 = j1 + bx * NB, nr = max(0, min(NB, n + 1 - r0));
        double accD[2][4][2], accX[2][4][2];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) accD[a][c][0] = accD[a][c][1] = accX[a][c][0] = accX[a][c][1] = 0.0;
        if (k > 0) {
            load_tile(T0, L, ldl, j0, jp0, nb);      // diagonal-block rows of panel k-1
            load_tile(T1, L, ldl, r0, jp0, nr);      // slab rows of panel k-1
            __syncthreads();
            mma_64(T0, T0, accD);
            mma_64(T1, T0, accX);
            __syncthreads();
        }
        // strip values minus the look-ahead update -> factor view Dg (T0) and slab view Xs (T1), stride LDX
        double *Dg = T0, *Xs = T1;
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int r = wm + 8 * a + r8, cc = wn + 8 * c + 2 * kq + q;
                    double d = (r == cc) ? 1.0 : 0.0, x = 0.0;
                    if (r < nb && cc <= r) d = L[(size_t)(j0 + r) * ldl + j0 + cc] - accD[a][c][q];
                    if (r < nr && cc < nb) x = L[(size_t)(r0 + r) * ldl + j0 + cc] - accX[a][c][q];
                    Dg[r * LDX + cc] = d;
                    Xs[r * LDX + cc] = x;
                }
        __syncthreads();
        chol_64(Dg, colbuf, pivs, rs, nb, &flag[2 * b], j0, bx == 0);
        if (bx == 0)
            for (int i = tid; i < NB * NB; i += 256) {
                const int r = i >> 6, c = i & 63;
                if (r < nb && c <= r) L[(size_t)(j0 + r) * ldl + j0 + c] = Dg[r * LDX + c];
            }
        if (nr <= 0) return;
        if (tid < nr) {
            double x[NB];
#pragma unroll
            for (int c = 0; c < NB; ++c) x[c] = Xs[tid * LDX + c];
            row_trsm(x, Dg, rs);
#pragma unroll
            for (int c = 0; c < NB; ++c) Xs[tid * LDX + c] = x[c];
        }
        __syncthreads();
        for (int i = tid; i < NB * NB; i += 256) {
            const int r = i >> 6, c = i & 63;
            if (r < nr && c < nb) L[(size_t)(r0 + r) * ldl + j0 + c] = Xs[r * LDX + c];
        }
        return;
    }
    bx -= nslab;
    if (bx < ntiles) {
        // ------------------------------ U: trailing tile (ti, tj), tj <= ti, with panel k-1 ------------------------------
        int ti = (int)((sqrt(8.0 * (double)bx + 1.0) - 1.0) * 0.5);
        while ((ti + 1) * (ti + 2) / 2 <= bx) ++ti;
        while (ti * (ti + 1) / 2 > bx) --ti;
        const int tj = bx - ti * (ti + 1) / 2;
        const int i0 = j1 + ti * NB, c0 = j1 + tj * NB;
        const int nri = max(0, min(NB, n + 1 - i0)), nrj = max(0, min(NB, n - c0));
        load_tile(T0, L, ldl, i0, jp0, nri);
        if (tj != ti) load_tile(T1, L, ldl, c0, jp0, nrj);
        __syncthreads();
        double acc[2][4][2];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][c][0] = acc[a][c][1] = 0.0;
        mma_64(T0, tj != ti ? T1 : T0, acc);
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int i = i0 + wm + 8 * a + r8, j = c0 + wn + 8 * c + 2 * kq;
                if (i > n) continue;
                double *dst = &L[(size_t)i * ldl + j];
                if (j + 1 < n && j + 1 <= i) {
                    double2 v = *reinterpret_cast<double2 *>(dst);
                    v.x -= acc[a][c][0]; v.y -= acc[a][c][1];
                    *reinterpret_cast<double2 *>(dst) = v;
                } else if (j < n && j <= i) {
                    dst[0] -= acc[a][c][0];
                }
            }
        return;
    }
    // ------------------------------ I: W = inverse of the diagonal block of panel kI ------------------------------
    {
        const int kI = (k < nblk) ? k - 1 : nblk - 1;       // the launch after the last panel inverts the last block
        const int q0 = kI * NB, nq = min(NB, n - q0);
        double *Dg = T0;
        for (int i = tid; i < NB * NB; i += 256) {
            const int r = i >> 6, c = i & 63;
            Dg[r * LDX + c] = (r < nq && c <= r) ? L[(size_t)(q0 + r) * ldl + q0 + c] : (r == c ? 1.0 : 0.0);
        }
        __syncthreads();
        if (tid < NB) rs[tid] = 1.0 / Dg[tid * LDX + tid];
        __syncthreads();
        double *W = Winv + ((size_t)b * nblk + kI) * NB * NB;
        if (tid < NB) {
            double x[NB];
#pragma unroll
            for (int c = 0; c < NB; ++c) x[c] = (c == tid) ? 1.0 : 0.0;
            row_trsm(x, Dg, rs);                    // x[c] = W[c][tid]
#pragma unroll
            for (int c = 0; c < NB; ++c) W[c * NB + tid] = x[c];
        }
    }
}

// Backward substitution L^T y = z (z = row n of Lf), c = D y.  One cluster of CS CTAs per system; CTA `rank`
// owns the 64-column blocks with block % CS == rank and keeps their part of z in shared memory.
__global__ void __cluster_dims__(CS, 1, 1) __launch_bounds__(256)
k_chol_backsolve(const double *__restrict__ Lf, const double *__restrict__ Winv, const double *__restrict__ dscale,
                 double *__restrict__ coef, int n, int ldl, int nblk) {
    extern __shared__ double zs[];                 // [nblk * 64] (own blocks valid)
    __shared__ double ybuf[2][NB];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), b = blockIdx.y, tid = threadIdx.x;
    const double *L = Lf + (size_t)b * (n + 1) * ldl;
    for (int i = tid; i < nblk * NB; i += 256) zs[i] = (i < n) ? L[(size_t)n * ldl + i] : 0.0;
    cluster.sync();
    for (int blk = nblk - 1; blk >= 0; --blk) {
        const int i0 = blk * NB, nbk = min(NB, n - i0);
        if (rank == blk % CS && tid < NB) {
            // y_i = sum_{k >= i} W[k][i] z_k
            const double *W = Winv + ((size_t)b * nblk + blk) * NB * NB;
            double y0 = 0.0, y1 = 0.0;
            for (int k = tid; k < nbk; k += 2) {   // two chains; entries above the diagonal of W are zero
                y0 = fma(W[k * NB + tid], zs[i0 + k], y0);
                if (k + 1 < nbk) y1 = fma(W[(k + 1) * NB + tid], zs[i0 + k + 1], y1);
            }
            const double y = y0 + y1;
            if (tid < nbk) coef[(size_t)b * n + i0 + tid] = y * dscale[(size_t)b * n + i0 + tid];
#pragma unroll
            for (int c = 0; c < CS; ++c) cluster.map_shared_rank(&ybuf[blk & 1][0], c)[tid] = (tid < nbk) ? y : 0.0;
        }
        cluster.sync();
        // z_j -= sum_k L[i0 + k][j] y_k for the columns of the blocks this CTA owns below blk (nearest first)
        const int col = tid & 63, slot = tid >> 6;
        const double *yb = ybuf[blk & 1];
        int first = blk - 1 - ((blk - 1 - rank) % CS + CS) % CS;      // largest owned block < blk
        for (int ob = first - slot * CS; ob >= 0; ob -= 4 * CS) {
            const double *src = L + (size_t)i0 * ldl + ob * NB + col;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int kk = 0;
            for (; kk + 4 <= nbk; kk += 4) {
                s0 = fma(src[(size_t)kk * ldl], yb[kk], s0);
                s1 = fma(src[(size_t)(kk + 1) * ldl], yb[kk + 1], s1);
                s2 = fma(src[(size_t)(kk + 2) * ldl], yb[kk + 2], s2);
                s3 = fma(src[(size_t)(kk + 3) * ldl], yb[kk + 3], s3);
            }
            for (; kk < nbk; ++kk) s0 = fma(src[(size_t)kk * ldl], yb[kk], s0);
            zs[ob * NB + col] -= (s0 + s1) + (s2 + s3);
        }
        __syncthreads();
    }
}

}  // namespace

int solve_num_blocks(int n) { return (n + NB - 1) / NB; }

cudaError_t launch_solve(sfft_plan *p, double *d_coef) {
    const int n = p->n, ldl = p->ldl, nbat = p->nbatch, nblk = solve_num_blocks(n);
    k_scale_diag<<<dim3((n + 255) / 256, nbat), 256, 0, p->stream>>>(p->M, p->dscale, p->flag, n);
    k_scale_copy<<<dim3((n + 127) / 128, n + 1, nbat), 128, 0, p->stream>>>(p->M, p->rhs, p->dscale, p->Lf, n, ldl);
    p->launches += 2;
    cudaError_t e = cudaFuncSetAttribute(k_chol_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStepSmem);
    if (e != cudaSuccess) return e;
    for (int k = 0; k <= nblk; ++k) {
        int nslab = 0, ntiles = 0;
        if (k < nblk) {
            const int j1 = std::min(n, (k + 1) * NB);
            nslab = (n + 1 - j1 + NB - 1) / NB;                       // rows j1..n (the rhs row is row n)
            if (k > 0) { const int nt = nslab; ntiles = nt * (nt + 1) / 2; }
        }
        const int grid = nslab + ntiles + (k > 0 ? 1 : 0);
        k_chol_step<<<dim3(grid, nbat), 256, kStepSmem, p->stream>>>(p->Lf, p->Winv, p->flag, n, ldl, k, nslab, ntiles, nblk);
        p->launches++;
    }
    const size_t smem = (size_t)nblk * NB * sizeof(double);
    e = cudaFuncSetAttribute(k_chol_backsolve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_chol_backsolve<<<dim3(CS, nbat), 256, smem, p->stream>>>(p->Lf, p->Winv, p->dscale, d_coef, n, ldl, nblk);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
