// Step a6: dense FP64 solve of the SPD normal system (DESIGN g11).
//
//   1. Jacobi scaling  A = D M D, D = diag(M)^-1/2  (removes the 10^6..10^12 spread between
//      kernel and background unknowns), rhs appended as an extra ROW of the lower triangle:
//      factoring [[A, .],[r^T D, .]] leaves z = L^-1 D r in that row, so the forward
//      substitution comes for free with the panel solves.
//   2. Right-looking blocked Cholesky, panel width NB: per panel one kernel factors the
//      diagonal block in shared memory and solves the panel rows (each CTA re-factors the
//      32x32 block instead of waiting on another launch), one kernel applies the symmetric
//      rank-NB update to the trailing lower triangle (64x64 register-tiled FP64 FMA).
//   3. Backward substitution L^T y = z in one CTA per system, c = D y.
// A non-positive pivot writes its index to flag[2*b] (reported as SFFT_ERR_NOT_SPD).
#include <algorithm>

#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int NB = 32;   // panel width
constexpr int TR = 64;   // panel rows per CTA in the triangular solve
constexpr int TS = 64;   // trailing-update tile

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

// Panel kernel for columns [j0, j0+nb): every CTA factors the diagonal block in shared memory,
// CTA 0 stores it, and each CTA solves X L11^T = A21 for its TR rows below the block.
__global__ void __launch_bounds__(256) k_chol_panel(double *__restrict__ Lf, int *flag, int n, int ldl, int j0) {
    __shared__ double A11[NB][NB + 1];
    __shared__ double X[TR][NB + 1];
    const int b = blockIdx.y, nb = min(NB, n - j0), tid = threadIdx.x;
    double *L = Lf + (size_t)b * (n + 1) * ldl;
    for (int i = tid; i < NB * NB; i += 256) {
        int r = i / NB, c = i % NB;
        A11[r][c] = (r < nb && c <= r) ? L[(size_t)(j0 + r) * ldl + j0 + c] : (r == c ? 1.0 : 0.0);
    }
    __syncthreads();
    for (int k = 0; k < nb; ++k) {
        double piv = A11[k][k];
        if (!(piv > 0.0)) {
            if (tid == 0 && blockIdx.x == 0) atomicCAS(&flag[2 * b], -1, j0 + k);
            piv = 1.0;
        }
        double s = sqrt(piv);
        __syncthreads();
        if (tid == 0) A11[k][k] = s;
        if (tid > k && tid < nb) A11[tid][k] /= s;
        __syncthreads();
        for (int i = tid; i < NB * NB; i += 256) {
            int r = i / NB, c = i % NB;
            if (c > k && r >= c && r < nb) A11[r][c] -= A11[r][k] * A11[c][k];
        }
        __syncthreads();
    }
    if (blockIdx.x == 0)
        for (int i = tid; i < NB * NB; i += 256) {
            int r = i / NB, c = i % NB;
            if (r < nb && c <= r) L[(size_t)(j0 + r) * ldl + j0 + c] = A11[r][c];
        }
    const int r0 = j0 + nb + blockIdx.x * TR;          // first row of this CTA's slab (rows up to n inclusive)
    const int nr = min(TR, n + 1 - r0);
    if (nr <= 0) return;
    for (int i = tid; i < TR * NB; i += 256) {
        int r = i / NB, c = i % NB;
        X[r][c] = (r < nr && c < nb) ? L[(size_t)(r0 + r) * ldl + j0 + c] : 0.0;
    }
    __syncthreads();
    if (tid < nr) {
        double x[NB];
#pragma unroll
        for (int c = 0; c < NB; ++c) x[c] = X[tid][c];
#pragma unroll
        for (int k = 0; k < NB; ++k) {
            double v = x[k];
#pragma unroll
            for (int m = 0; m < k; ++m) v = fma(-x[m], A11[k][m], v);
            x[k] = v / A11[k][k];
        }
#pragma unroll
        for (int c = 0; c < NB; ++c) X[tid][c] = x[c];
    }
    __syncthreads();
    for (int i = tid; i < TR * NB; i += 256) {
        int r = i / NB, c = i % NB;
        if (r < nr && c < nb) L[(size_t)(r0 + r) * ldl + j0 + c] = X[r][c];
    }
}

// Trailing update C[i][j] -= sum_k P[i][k] P[j][k] over the lower triangle of rows/cols >= j1,
// P = panel columns [j0, j0+nb).  One CTA per 64x64 tile (lower-triangular tile index), 4x4 per thread.
__global__ void __launch_bounds__(256) k_chol_syrk(double *__restrict__ Lf, int n, int ldl, int j0, int nb, int j1) {
    __shared__ double Pi[NB][TS + 1];
    __shared__ double Pj[NB][TS + 1];
    const int b = blockIdx.y;
    // blockIdx.x -> (ti, tj), tj <= ti
    int ti = (int)((sqrt(8.0 * (double)blockIdx.x + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= (int)blockIdx.x) ++ti;
    while (ti * (ti + 1) / 2 > (int)blockIdx.x) --ti;
    const int tj = blockIdx.x - ti * (ti + 1) / 2;
    double *L = Lf + (size_t)b * (n + 1) * ldl;
    const int i0 = j1 + ti * TS, c0 = j1 + tj * TS, tid = threadIdx.x;
    for (int i = tid; i < TS * NB; i += 256) {
        int r = i / NB, k = i % NB;
        Pi[k][r] = (i0 + r <= n && k < nb) ? L[(size_t)(i0 + r) * ldl + j0 + k] : 0.0;
        Pj[k][r] = (c0 + r < n && k < nb) ? L[(size_t)(c0 + r) * ldl + j0 + k] : 0.0;
    }
    __syncthreads();
    const int tx = tid % 16, ty = tid / 16;
    double acc[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[a][c] = 0.0;
#pragma unroll 8
    for (int k = 0; k < NB; ++k) {
        double pi[4], pj[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) { pi[a] = Pi[k][ty + 16 * a]; pj[a] = Pj[k][tx + 16 * a]; }
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][c] = fma(pi[a], pj[c], acc[a][c]);
    }
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            int i = i0 + ty + 16 * a, j = c0 + tx + 16 * c;
            if (i <= n && j < n && j <= i) L[(size_t)i * ldl + j] -= acc[a][c];
        }
}

// Backward substitution L^T y = z (z = row n of Lf), c = D y.  One CTA (512 threads) per system,
// blocks of 32 unknowns from the bottom: a warp solves the 32x32 triangle, then all threads
// update the remaining right-hand side (coalesced along the row of L).
__global__ void __launch_bounds__(512) k_chol_backsolve(const double *__restrict__ Lf, const double *__restrict__ dscale,
                                                        double *__restrict__ coef, int n, int ldl) {
    extern __shared__ double z[];     // [n]
    __shared__ double yb[32];
    const int b = blockIdx.x, tid = threadIdx.x;
    const double *L = Lf + (size_t)b * (n + 1) * ldl;
    for (int i = tid; i < n; i += blockDim.x) z[i] = L[(size_t)n * ldl + i];
    __syncthreads();
    for (int i1 = n; i1 > 0; i1 -= 32) {
        const int i0 = max(0, i1 - 32), nbk = i1 - i0;
        if (tid < 32) {
            // y_i = (z_i - sum_{k>i in block} L[k][i] y_k) / L[i][i], solved from the bottom.
            // Lane `tid` first pulls column tid of the 32x32 block into registers (one round trip).
            double lc[32];
#pragma unroll
            for (int k = 0; k < 32; ++k)
                lc[k] = (k < nbk && tid <= k) ? L[(size_t)(i0 + k) * ldl + i0 + tid] : (k == tid ? 1.0 : 0.0);
            double zi = tid < nbk ? z[i0 + tid] : 0.0;
#pragma unroll
            for (int k = 31; k >= 0; --k) {
                double dk = __shfl_sync(0xffffffffu, lc[k], k);
                double yk = __shfl_sync(0xffffffffu, zi, k) / dk;
                if (tid == k) zi = yk;
                else if (tid < k) zi = fma(-lc[k], yk, zi);
            }
            if (tid < nbk) { yb[tid] = zi; z[i0 + tid] = zi; }
        }
        __syncthreads();
        for (int j = tid; j < i0; j += blockDim.x) {
            double s = z[j];
            for (int k = 0; k < nbk; ++k) s = fma(-L[(size_t)(i0 + k) * ldl + j], yb[k], s);
            z[j] = s;
        }
        __syncthreads();
    }
    for (int i = tid; i < n; i += blockDim.x) coef[(size_t)b * n + i] = z[i] * dscale[(size_t)b * n + i];
}

}  // namespace

cudaError_t launch_solve(sfft_plan *p, double *d_coef) {
    const int n = p->n, ldl = p->ldl, nbat = p->nbatch;
    k_scale_diag<<<dim3((n + 255) / 256, nbat), 256, 0, p->stream>>>(p->M, p->dscale, p->flag, n);
    k_scale_copy<<<dim3((n + 127) / 128, n + 1, nbat), 128, 0, p->stream>>>(p->M, p->rhs, p->dscale, p->Lf, n, ldl);
    p->launches += 2;
    for (int j0 = 0; j0 < n; j0 += NB) {
        const int nb = std::min(NB, n - j0), j1 = j0 + nb;
        const int rows_below = n + 1 - j1;                        // includes the appended rhs row
        const int nslab = std::max(1, (rows_below + TR - 1) / TR);
        k_chol_panel<<<dim3(nslab, nbat), 256, 0, p->stream>>>(p->Lf, p->flag, n, ldl, j0);
        p->launches++;
        if (j1 < n) {
            const int nt = (rows_below + TS - 1) / TS;
            k_chol_syrk<<<dim3(nt * (nt + 1) / 2, nbat), 256, 0, p->stream>>>(p->Lf, n, ldl, j0, nb, j1);
            p->launches++;
        }
    }
    size_t smem = (size_t)n * sizeof(double);
    cudaError_t e = cudaFuncSetAttribute(k_chol_backsolve, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_chol_backsolve<<<nbat, 512, smem, p->stream>>>(p->Lf, p->dscale, d_coef, n, ldl);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
