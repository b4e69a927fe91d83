// Step a6: dense FP64 solve of the SPD normal system (DESIGN g11).
//
//   1. Jacobi scaling  A = D M D, D = diag(M)^-1/2  (removes the 10^6..10^12 spread between
//      kernel and background unknowns), rhs appended as an extra ROW of the lower triangle:
//      factoring [[A, .],[r^T D, .]] leaves z = L^-1 D r in that row, so the forward
//      substitution comes for free with the panel solves.
//   2. Right-looking blocked Cholesky with one look-ahead step, panel width NB = 64, ONE launch
//      per panel (k_chol_step).  Launch k holds two kinds of CTA:
//        P  (one per 64-row slab below the diagonal block of panel k): applies panel k-1 to its
//           rows of column strip k and to the diagonal block (FP64 tensor cores), factors the
//           64x64 diagonal block together with the inverse W of its factor (every P CTA redundantly -
//           cheaper than another launch), and solves its slab as the dense contraction X = S W^T;
//        U  (one per 64x64 tile of the lower triangle right of strip k): rank-64 update with
//           panel k-1 on the FP64 tensor cores (mma.sync.m8n8k4.f64: a dense contraction).
//      P(k) needs only panel k-1 and the U updates of launch k-1, so the latency-bound panel
//      chain (factor + triangular solve) overlaps the throughput-bound trailing update.
//      Throughput regime (many trailing tiles: batches, n in the thousands): three launches per panel
//      instead - one factoring CTA per system (k_chol_step with a single slab), lean slab CTAs that read
//      W from global memory (k_chol_slab), and the trailing update by segments of tile rows with a
//      cp.async double buffer and register-prefetched C tiles (k_chol_update_row).
//   3. Backward substitution L^T y = z with one CTA per 64-column block: CTA b prefetches its tiles of the factor,
//      consumes the blocks y_j (j > b) as their owners publish them in global memory (the values are their own
//      flags: a sentinel pattern marks "not yet written"), then forms y_b = W_b^T z_b with W_b = L_bb^-1 from the
//      factorisation.  c = D y.
// A diagonal entry that is not positive and finite, or a pivot of the scaled matrix (unit diagonal) that is not
// finite or lies below kPivotFloor * n (rounding-noise level of the assembled entries: the system is numerically
// rank-deficient even where the noise happens to be positive), writes its index to flag[2*b] (SFFT_ERR_NOT_SPD).
#include <cuda.h>          // CUtensorMap (types only: the encoder is fetched through cudaGetDriverEntryPoint)

#include <algorithm>

#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int NB = 64;        // panel width = tile size
constexpr int LDT = NB + 4;   // smem stride of MMA operand tiles (= 4 mod 16: conflict-free fragments)
constexpr int LDX = NB + 1;   // smem stride of the factor / solve views (conflict-free row-per-thread access)
constexpr double kPivotFloor = 64.0 * 2.220446049250313e-16;   // x n: smallest pivot of the scaled matrix taken as non-zero

__device__ __forceinline__ bool pivot_ok(double p, double pmin) { return p > pmin && p < 1e300; }

__global__ void k_scale_diag(const double *__restrict__ M, double *__restrict__ dscale, int *flag, int n,
                             unsigned long long *__restrict__ ybuf, int ny, unsigned long long sentinel, int *ticket) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
    if (i == 0 && b == 0) *ticket = 0;                     // start-order counter of the look-back back substitution
    if (i < ny) ybuf[(size_t)b * ny + i] = sentinel;       // "not yet published" marks of the look-back back substitution
    if (i >= n) return;
    double d = M[((size_t)b * n + i) * n + i];
    if (!(d > 0.0 && d < 1e300)) { atomicCAS(&flag[2 * b], -1, i); d = 1.0; }
    dscale[(size_t)b * n + i] = rsqrt(d);
}

// Lf[i][j] = M[i][j] d_i d_j (j <= i), row n = rhs_j d_j.  CTA = 16 rows x 128 columns, thread = 4 rows x 2 columns
// (eight independent loads in flight); tiles above the diagonal exit at once.
__global__ void __launch_bounds__(256) k_scale_copy(const double *__restrict__ M, const double *__restrict__ rhs,
                                                    const double *__restrict__ dscale, double *__restrict__ Lf, int n, int ldl) {
    const int j = blockIdx.x * 128 + 2 * (threadIdx.x & 63), i0 = blockIdx.y * 16 + (threadIdx.x >> 6), b = blockIdx.z;
    if (blockIdx.x * 128 > blockIdx.y * 16 + 15 || j >= n) return;
    const double *d = dscale + (size_t)b * n;
    const double dj0 = d[j], dj1 = (j + 1 < n) ? d[j + 1] : 0.0;
    double v0[4], v1[4], di[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int i = i0 + 4 * r;
        v0[r] = v1[r] = 0.0; di[r] = 1.0;
        if (i < n) {
            const double *src = M + ((size_t)b * n + i) * n + j;
            di[r] = d[i];
            if (j <= i) v0[r] = src[0];
            if (j + 1 <= i) v1[r] = src[1];
        } else if (i == n) {
            v0[r] = rhs[(size_t)b * n + j];
            if (j + 1 < n) v1[r] = rhs[(size_t)b * n + j + 1];
        }
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int i = i0 + 4 * r;
        if (i > n || j > i) continue;
        double *dst = Lf + ((size_t)b * (n + 1) + i) * ldl + j;
        if (j + 1 <= i && j + 1 < n) *reinterpret_cast<double2 *>(dst) = make_double2(v0[r] * di[r] * dj0, v1[r] * di[r] * dj1);
        else dst[0] = v0[r] * di[r] * dj0;
    }
}

// T[r][c] = L[row0 + r][col0 + c] for r < nr (else 0), 64 columns, into an MMA operand tile (stride LDT).
// Split in an issue half (all global loads in flight at once) and a store half.
struct TileRegs { double2 v[NB * NB / 2 / 256]; };
__device__ __forceinline__ void tile_fetch(TileRegs &t, const double *L, int ldl, int row0, int col0, int nr) {
#pragma unroll
    for (int q = 0; q < NB * NB / 2 / 256; ++q) {
        const int i = threadIdx.x + 256 * q, r = i >> 5, c = (i & 31) * 2;
        t.v[q] = make_double2(0.0, 0.0);
        if (r < nr) t.v[q] = *reinterpret_cast<const double2 *>(&L[(size_t)(row0 + r) * ldl + col0 + c]);
    }
}
__device__ __forceinline__ void tile_store(double *T, const TileRegs &t) {
#pragma unroll
    for (int q = 0; q < NB * NB / 2 / 256; ++q) {
        const int i = threadIdx.x + 256 * q, r = i >> 5, c = (i & 31) * 2;
        T[r * LDT + c] = t.v[q].x;
        T[r * LDT + c + 1] = t.v[q].y;
    }
}

// 1/x to full double precision for normal positive x: MUFU seed + two Newton steps (no slow-path call)
__device__ __forceinline__ double fast_rcp(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
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

// acc += A W^T for a LOWER-TRIANGULAR right operand W (64x64 tiles, stride LDT): column tile ct of the product
// only needs k < 8 ct + 8, so each warp takes the column tiles {0,3,4,7} (HALF 0) or {1,2,5,6} (HALF 1) - 18 of
// the 36 live (tile, k-block) pairs each, against 32 for the dense product.  Rows as in mma_64.
// acc[a][c][q] <-> row 16*(w>>1) + 8a + (lane>>2), col 8*ct(c) + 2*(lane&3) + q
template <int HALF>
__device__ __forceinline__ int lower_tile(int c) { return HALF == 0 ? (c == 0 ? 0 : c == 1 ? 3 : c == 2 ? 4 : 7) : (c == 0 ? 1 : c == 1 ? 2 : c == 2 ? 5 : 6); }
template <int HALF>
__device__ __forceinline__ void mma_64_lowerB(const double *A, const double *W, double (&acc)[2][4][2]) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, r = lane >> 2, kq = lane & 3;
    const double *ap = A + ((warp >> 1) * 16 + r) * LDT + kq;
    const double *bp = W + r * LDT + kq;
#pragma unroll
    for (int k = 0; k < NB; k += 4) {
        double af[2];
#pragma unroll
        for (int a = 0; a < 2; ++a) af[a] = ap[a * 8 * LDT + k];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int ct = lower_tile<HALF>(c);
            if (k < 8 * ct + 8) {                    // compile-time after unrolling
                const double bf = bp[ct * 8 * LDT + k];
#pragma unroll
                for (int a = 0; a < 2; ++a) dmma884(acc[a][c], af[a], bf);
            }
        }
    }
}

// acc += A A^T restricted to the lower triangle (tile granularity 8): warp (RB, HALF) owns the row tiles {RB, 7-RB}
// and the column tiles of lower_tile<HALF>, so every warp carries 4 or 5 live tiles of the 36 (8 for the dense
// product).  acc[a][c][q] <-> row 8*rt(a) + (lane>>2), col 8*ct(c) + 2*(lane&3) + q, rt(0) = RB, rt(1) = 7 - RB.
template <int RB, int HALF>
__device__ __forceinline__ void mma_64_symlower(const double *A, double (&acc)[2][4][2]) {
    const int lane = threadIdx.x & 31, r = lane >> 2, kq = lane & 3;
    const double *ap = A + r * LDT + kq;
#pragma unroll 4
    for (int k = 0; k < NB; k += 4) {
        const double a0 = ap[RB * 8 * LDT + k], a1 = ap[(7 - RB) * 8 * LDT + k];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int ct = lower_tile<HALF>(c);
            if (ct <= 7 - RB) {                       // compile-time
                const double bf = ap[ct * 8 * LDT + k];
                if (ct <= RB) dmma884(acc[0][c], a0, bf);
                dmma884(acc[1][c], a1, bf);
            }
        }
    }
}
__device__ __forceinline__ void mma_64_symlower_dispatch(const double *A, double (&acc)[2][4][2]) {
    switch (threadIdx.x >> 5) {          // warp-uniform
        case 0: mma_64_symlower<0, 0>(A, acc); break;
        case 1: mma_64_symlower<0, 1>(A, acc); break;
        case 2: mma_64_symlower<1, 0>(A, acc); break;
        case 3: mma_64_symlower<1, 1>(A, acc); break;
        case 4: mma_64_symlower<2, 0>(A, acc); break;
        case 5: mma_64_symlower<2, 1>(A, acc); break;
        case 6: mma_64_symlower<3, 0>(A, acc); break;
        default: mma_64_symlower<3, 1>(A, acc); break;
    }
}

// In-place Cholesky of the 64x64 block Dg (shared memory, stride LDX, lower triangle valid, identity
// padded beyond nb) by all 256 threads, together with the inverse of its factor: the elimination is
// run on the augmented block [A | I], which turns I into W = L^-1.  Every thread keeps 4x4 register
// tiles of A and of the augmented part (rows ty+16a, cols tx+16b); step k publishes column k of A and
// row k of the augmented part through double-buffered shared vectors, so there is ONE barrier per
// column; the scalings by 1/sqrt(pivot) are deferred to the end.
// On exit: Wt[r*LDT + c] = W[r][c] (an MMA operand tile; may alias Dg) and, when `store` is set, W goes
// to Wg (64x64, row-major).  The factor's diagonal block itself is NOT written back: nothing downstream
// reads it (the back substitution uses W), and the other P CTAs of this launch - which may be scheduled
// after this one has finished when the grid exceeds one wave - still read the unfactored block from Lf.
__device__ __forceinline__ void chol_inv_64(const double *Dg, double *Wt, double *colbuf, double *rowbuf, double *pivs,
                                            double *rs, int nb, int *flag, int gidx0, bool store, double *Wg, double pmin) {
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    double t[4][4], e[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            t[a][b] = Dg[(ty + 16 * a) * LDX + tx + 16 * b];
            e[a][b] = (a == b && tx == ty) ? 1.0 : 0.0;
        }
#pragma unroll
    for (int b = 0; b < 4; ++b) {
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            const int k = 16 * b + kk;
            if (k >= nb) break;                              // uniform
            double *cb = colbuf + (k & 1) * NB, *rb = rowbuf + (k & 1) * NB;
            if (tx == kk) {
#pragma unroll
                for (int a = b; a < 4; ++a) cb[ty + 16 * a] = t[a][b];      // rows above the block are never read
            }
            if (ty == kk) {
#pragma unroll
                for (int bb = 0; bb <= b; ++bb) rb[tx + 16 * bb] = e[b][bb];  // E is lower triangular
            }
            __syncthreads();
            // the pivot test is taken off the per-column chain: pivots are recorded and checked once after the
            // loop (a non-positive pivot makes everything after it garbage, which is reported, not used)
            const double piv = cb[k];
            if (tid == 0) pivs[k] = piv;
            const double inv = fast_rcp(piv);
            // only the lower sub-blocks (a >= bb >= b) are ever read: the step is bound by FP64 issue
            // (two warps per scheduler, two cycles per FP64 warp instruction), so the dead upper ones are skipped
            double lr[4];
#pragma unroll
            for (int a = b; a < 4; ++a) lr[a] = cb[ty + 16 * a] * inv;
#pragma unroll
            for (int bb = b; bb < 4; ++bb) {
                const double lc = cb[tx + 16 * bb];
                if (bb > b || tx > kk) {
#pragma unroll
                    for (int a = bb; a < 4; ++a) t[a][bb] = fma(-lr[a], lc, t[a][bb]);
                }
            }
#pragma unroll
            for (int bb = 0; bb <= b; ++bb) {
                const double ec = rb[tx + 16 * bb];
#pragma unroll
                for (int a = b; a < 4; ++a)
                    if (a > b || ty > kk) e[a][bb] = fma(-lr[a], ec, e[a][bb]);
            }
        }
    }
    __syncthreads();       // Dg fully consumed (registers), pivs complete
    if (store && tid < nb && !pivot_ok(pivs[tid], pmin)) {
        // first failing column of this block: the lowest index wins; an earlier block's failure (already in
        // the flag from a previous launch) is kept by the compare-and-swap on -1 only
        bool first = true;
        for (int q = 0; q < tid; ++q) first = first && pivot_ok(pivs[q], pmin);
        if (first) atomicCAS(flag, -1, gidx0 + tid);
    }
    if (tid < NB) rs[tid] = (tid < nb) ? rsqrt(pivs[tid]) : 1.0;
    __syncthreads();
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int r = ty + 16 * a, c = tx + 16 * b;
            const double w = e[a][b] * rs[r];
            Wt[r * LDT + c] = w;
            if (store) Wg[r * NB + c] = w;
        }
    __syncthreads();
}

// U: rank-64 update of trailing tile `bx` = (ti, tj), tj <= ti, of the lower triangle right of strip k with
// panel k-1 (columns jp0..jp0+63); j1 = first row/column after strip k.  T0, T1: MMA operand tiles.
__device__ __forceinline__ void chol_update_tile(double *__restrict__ L, int ldl, int n, int j1, int jp0, int bx,
                                                 double *T0, double *T1) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r8 = lane >> 2, kq = lane & 3, wm = (warp >> 1) * 16, wn = (warp & 1) * 32;
    int ti = (int)((sqrt(8.0 * (double)bx + 1.0) - 1.0) * 0.5);
    while ((ti + 1) * (ti + 2) / 2 <= bx) ++ti;
    while (ti * (ti + 1) / 2 > bx) --ti;
    const int tj = bx - ti * (ti + 1) / 2;
    const int i0 = j1 + ti * NB, c0 = j1 + tj * NB;
    const int nri = max(0, min(NB, n + 1 - i0)), nrj = max(0, min(NB, n - c0));
    {
        TileRegs ta;
        tile_fetch(ta, L, ldl, i0, jp0, nri);
        tile_store(T0, ta);
        if (tj != ti) {
            tile_fetch(ta, L, ldl, c0, jp0, nrj);
            tile_store(T1, ta);
        }
    }
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
}

constexpr size_t kStepSmem = (size_t)(2 * NB * LDT + 4 * NB + NB + NB) * sizeof(double);
constexpr size_t kUpdSmem = (size_t)(2 * NB * LDT) * sizeof(double);
constexpr size_t kRowSmem = (size_t)(3 * NB * LDT) * sizeof(double);

// One launch per panel k (see the header).  grid.x = nslab P CTAs, then ntiles U CTAs (k >= 1).
__global__ void __launch_bounds__(256) k_chol_step(double *__restrict__ Lf, double *__restrict__ Winv, int *flag, int n,
                                                   int ldl, int k, int nslab, int ntiles, int nblk) {
    // programmatic dependent launch: this grid may be scheduled while the previous panel's grid drains; nothing
    // of the previous grid is read before the wait, and the next grid may be scheduled from here on
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;");
    extern __shared__ double sm[];
    double *T0 = sm, *T1 = sm + NB * LDT;                   // MMA operand tiles; later the factor / slab views
    double *colbuf = sm + 2 * NB * LDT, *rowbuf = colbuf + 2 * NB, *pivs = rowbuf + 2 * NB, *rs = pivs + NB;
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
        // strip values (diagonal block and slab rows of strip k) in MMA fragment layout, fetched up front
        double dv[2][4][2], xv[2][4][2];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int r = wm + 8 * a + r8, cc = wn + 8 * c + 2 * kq + q;
                    // diagonal block in the layout of mma_64_symlower (row tiles {rb, 7-rb}, interleaved column tiles)
                    const int rd = 8 * (a == 0 ? (warp >> 1) : 7 - (warp >> 1)) + r8;
                    const int cd = 8 * ((warp & 1) ? lower_tile<1>(c) : lower_tile<0>(c)) + 2 * kq + q;
                    dv[a][c][q] = (rd < nb && cd <= rd) ? L[(size_t)(j0 + rd) * ldl + j0 + cd] : ((rd == cd) ? 1.0 : 0.0);
                    xv[a][c][q] = (r < nr && cc < nb) ? L[(size_t)(r0 + r) * ldl + j0 + cc] : 0.0;
                }
        if (k > 0) {
            TileRegs td, ts;
            tile_fetch(td, L, ldl, j0, jp0, nb);     // diagonal-block rows of panel k-1
            tile_fetch(ts, L, ldl, r0, jp0, nr);     // slab rows of panel k-1
            tile_store(T0, td);
            tile_store(T1, ts);
            __syncthreads();
            mma_64_symlower_dispatch(T0, accD);
            mma_64(T1, T0, accX);
            __syncthreads();
        }
        // strip values minus the look-ahead update -> factor view Dg (T0, stride LDX) and slab operand tile S (T1)
        double *Dg = T0, *St = T1;
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int r = wm + 8 * a + r8, cc = wn + 8 * c + 2 * kq + q;
                    const int rd = 8 * (a == 0 ? (warp >> 1) : 7 - (warp >> 1)) + r8;
                    const int cd = 8 * ((warp & 1) ? lower_tile<1>(c) : lower_tile<0>(c)) + 2 * kq + q;
                    const bool dl = (rd < nb && cd <= rd), xl = (r < nr && cc < nb);
                    Dg[rd * LDX + cd] = dl ? dv[a][c][q] - accD[a][c][q] : dv[a][c][q];
                    St[r * LDT + cc] = xl ? xv[a][c][q] - accX[a][c][q] : 0.0;
                }
        __syncthreads();
        // factor the diagonal block and invert its factor; W replaces Dg in T0 as an MMA operand tile
        chol_inv_64(Dg, T0, colbuf, rowbuf, pivs, rs, nb, &flag[2 * b], j0, bx == 0,
                    Winv + ((size_t)b * nblk + k) * NB * NB, kPivotFloor * n);
        if (nr <= 0) return;
        // slab solve X L11^T = S as the dense contraction X = S W^T
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) accX[a][c][0] = accX[a][c][1] = 0.0;
        if (warp & 1) mma_64_lowerB<1>(St, T0, accX); else mma_64_lowerB<0>(St, T0, accX);
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int ct = (warp & 1) ? lower_tile<1>(c) : lower_tile<0>(c);
                const int r = wm + 8 * a + r8, cc = 8 * ct + 2 * kq;
                if (r >= nr) continue;
                double *dst = &L[(size_t)(r0 + r) * ldl + j0 + cc];
                if (cc + 1 < nb) *reinterpret_cast<double2 *>(dst) = make_double2(accX[a][c][0], accX[a][c][1]);
                else if (cc < nb) dst[0] = accX[a][c][0];
            }
        return;
    }
    bx -= nslab;
    if (bx < ntiles) chol_update_tile(L, ldl, n, j1, jp0, bx, T0, T1);
}

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(a), "l"(gmem));
}

// T[r][0..63] = L[row0 + r][col0 ..] for r < nr (else 0) by asynchronous 16-byte copies (stride LDT)
__device__ __forceinline__ void tile_fetch_async(double *T, const double *L, int ldl, int row0, int col0, int nr) {
    if (nr == NB) {                      // full tile: one address, constant strides
        const int r = threadIdx.x >> 5, c = (threadIdx.x & 31) * 2;
        const double *src = L + (size_t)(row0 + r) * ldl + col0 + c;
        double *dst = T + r * LDT + c;
#pragma unroll
        for (int q = 0; q < NB * NB / 2 / 256; ++q) cp_async16(dst + 8 * q * LDT, src + (size_t)8 * q * ldl);
        asm volatile("cp.async.commit_group;");
        return;
    }
#pragma unroll
    for (int q = 0; q < NB * NB / 2 / 256; ++q) {
        const int i = threadIdx.x + 256 * q, r = i >> 5, c = (i & 31) * 2;
        if (r < nr) cp_async16(&T[r * LDT + c], &L[(size_t)(row0 + r) * ldl + col0 + c]);
        else { T[r * LDT + c] = 0.0; T[r * LDT + c + 1] = 0.0; }
    }
    asm volatile("cp.async.commit_group;");
}

// Trailing update, throughput regime: one CTA per tile ROW ti of the lower triangle right of strip k.  The row's
// own panel rows stay in shared memory; the column operands A_tj stream through a double buffer (cp.async) and
// the C tile is fetched into registers before the MMAs, so loads of tile tj+1 overlap the MMAs of tile tj.
// Rows are cut into segments of kRowSeg tiles so that work units are balanced; grid.x = number of segments
// (long rows first), grid.y = batch.
constexpr int kRowSeg = 16;
__host__ __device__ inline int row_segments(int nslab) {
    int s = 0;
    for (int ti = 0; ti < nslab; ++ti) s += (ti + kRowSeg) / kRowSeg;
    return s;
}
__global__ void __launch_bounds__(256, 2) k_chol_update_row(double *__restrict__ Lf, int n, int ldl, int k, int nslab) {
    extern __shared__ double sm[];
    double *Ti = sm, *Tj0 = sm + NB * LDT, *Tj1 = sm + 2 * NB * LDT;
    double *L = Lf + (size_t)blockIdx.y * (n + 1) * ldl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r8 = lane >> 2, kq = lane & 3, wm = (warp >> 1) * 16, wn = (warp & 1) * 32;
    const int j0 = k * NB, nb = min(NB, n - j0), j1 = j0 + nb, jp0 = j0 - NB;
    int ti = nslab - 1, seg = blockIdx.x;
    for (;;) {
        const int ns = (ti + kRowSeg) / kRowSeg;
        if (seg < ns) break;
        seg -= ns;
        --ti;
    }
    const int i0 = j1 + ti * NB, tj0 = seg * kRowSeg, tj1 = min(ti, tj0 + kRowSeg - 1);     // tiles tj0..tj1 of row ti
    const int nri = max(0, min(NB, n + 1 - i0));
    if (nri <= 0) return;
    tile_fetch_async(Ti, L, ldl, i0, jp0, nri);
    if (tj0 < ti) tile_fetch_async((tj0 & 1) ? Tj1 : Tj0, L, ldl, j1 + tj0 * NB, jp0, max(0, min(NB, n - (j1 + tj0 * NB))));
    // interior tiles (strictly below the diagonal, every row and column inside the system): no bounds tests, addresses
    // from two hoisted row pointers - the per-tile instruction overhead decides how well the two resident CTAs keep the
    // tensor pipe busy
    const bool rows_full = (i0 + NB <= n + 1);
    double *crow0 = L + (size_t)(i0 + wm + r8) * ldl + wn + 2 * kq, *crow1 = crow0 + (size_t)8 * ldl;
    for (int tj = tj0; tj <= tj1; ++tj) {
        const int c0 = j1 + tj * NB;
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                 // tile tj (and Ti) visible; MMAs of tile tj-1 done by every warp
        if (tj + 1 <= tj1 && tj + 1 < ti)
            tile_fetch_async((tj & 1) ? Tj0 : Tj1, L, ldl, c0 + NB, jp0, max(0, min(NB, n - (c0 + NB))));
        const bool interior = rows_full && tj < ti && c0 + NB <= n;
        // C tile into registers ahead of the MMAs
        double2 cv[2][4];
        if (interior) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                cv[0][c] = *reinterpret_cast<const double2 *>(crow0 + c0 + 8 * c);
                cv[1][c] = *reinterpret_cast<const double2 *>(crow1 + c0 + 8 * c);
            }
        } else {
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int i = i0 + wm + 8 * a + r8, j = c0 + wn + 8 * c + 2 * kq;
                    cv[a][c] = make_double2(0.0, 0.0);
                    if (i <= n && j + 1 < n && j + 1 <= i) cv[a][c] = *reinterpret_cast<const double2 *>(&L[(size_t)i * ldl + j]);
                    else if (i <= n && j < n && j <= i) cv[a][c].x = L[(size_t)i * ldl + j];
                }
        }
        double acc[2][4][2];
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[a][c][0] = acc[a][c][1] = 0.0;
        mma_64(Ti, tj == ti ? Ti : ((tj & 1) ? Tj1 : Tj0), acc);
        if (interior) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                *reinterpret_cast<double2 *>(crow0 + c0 + 8 * c) = make_double2(cv[0][c].x - acc[0][c][0], cv[0][c].y - acc[0][c][1]);
                *reinterpret_cast<double2 *>(crow1 + c0 + 8 * c) = make_double2(cv[1][c].x - acc[1][c][0], cv[1][c].y - acc[1][c][1]);
            }
        } else {
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int i = i0 + wm + 8 * a + r8, j = c0 + wn + 8 * c + 2 * kq;
                    if (i > n) continue;
                    double *dst = &L[(size_t)i * ldl + j];
                    if (j + 1 < n && j + 1 <= i) *reinterpret_cast<double2 *>(dst) = make_double2(cv[a][c].x - acc[a][c][0], cv[a][c].y - acc[a][c][1]);
                    else if (j < n && j <= i) dst[0] = cv[a][c].x - acc[a][c][0];
                }
        }
    }
}

// Slab CTAs of launch k without the diagonal-block factorisation (throughput regime): slab `1 + blockIdx.x`
// applies panel k-1 to its 64 rows of strip k and multiplies by W^T, with W = L_kk^-1 read from Winv (written
// by the one k_chol_step CTA per system launched just before).  grid.x = nslab - 1, grid.y = batch.
__global__ void __launch_bounds__(256, 2) k_chol_slab(double *__restrict__ Lf, const double *__restrict__ Winv, int n,
                                                      int ldl, int k, int nblk) {
    extern __shared__ double sm[];
    double *T0 = sm, *T1 = sm + NB * LDT;
    const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r8 = lane >> 2, kq = lane & 3, wm = (warp >> 1) * 16, wn = (warp & 1) * 32;
    double *L = Lf + (size_t)b * (n + 1) * ldl;
    const int j0 = k * NB, nb = min(NB, n - j0), j1 = j0 + nb, jp0 = j0 - NB;
    const int r0 = j1 + (blockIdx.x + 1) * NB, nr = max(0, min(NB, n + 1 - r0));
    if (nr <= 0) return;
    double acc[2][4][2], xv[2][4][2];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int r = wm + 8 * a + r8, cc = wn + 8 * c + 2 * kq + q;
                acc[a][c][q] = 0.0;
                xv[a][c][q] = (r < nr && cc < nb) ? L[(size_t)(r0 + r) * ldl + j0 + cc] : 0.0;
            }
    if (k > 0) {
        TileRegs t;
        tile_fetch(t, L, ldl, j0, jp0, nb);      // diagonal-block rows of panel k-1
        tile_store(T0, t);
        tile_fetch(t, L, ldl, r0, jp0, nr);      // slab rows of panel k-1
        tile_store(T1, t);
        __syncthreads();
        mma_64(T1, T0, acc);
        __syncthreads();
    }
    // S = strip values minus the look-ahead update (operand tile T1); W (operand tile T0)
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int r = wm + 8 * a + r8, cc = wn + 8 * c + 2 * kq + q;
                T1[r * LDT + cc] = (r < nr && cc < nb) ? xv[a][c][q] - acc[a][c][q] : 0.0;
                acc[a][c][q] = 0.0;
            }
    {
        const double *W = Winv + ((size_t)b * nblk + k) * NB * NB;
#pragma unroll
        for (int q = 0; q < NB * NB / 2 / 256; ++q) {
            const int i = tid + 256 * q, r = i >> 5, c = (i & 31) * 2;
            const double2 v = *reinterpret_cast<const double2 *>(&W[r * NB + c]);
            T0[r * LDT + c] = v.x;
            T0[r * LDT + c + 1] = v.y;
        }
    }
    __syncthreads();
    if (warp & 1) mma_64_lowerB<1>(T1, T0, acc); else mma_64_lowerB<0>(T1, T0, acc);
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int ct = (warp & 1) ? lower_tile<1>(c) : lower_tile<0>(c);
            const int r = wm + 8 * a + r8, cc = 8 * ct + 2 * kq;
            if (r >= nr) continue;
            double *dst = &L[(size_t)(r0 + r) * ldl + j0 + cc];
            if (cc + 1 < nb) *reinterpret_cast<double2 *>(dst) = make_double2(acc[a][c][0], acc[a][c][1]);
            else if (cc < nb) dst[0] = acc[a][c][0];
        }
}

// Backward substitution L^T y = z (z = row n of Lf), c = D y, look-back form.  One CTA per 64-column block b of one
// system; CTA b keeps z_b, prefetches the tiles L[j-rows][b-columns] of the blocks j > b through a ring of
// cp.async stages (the factor is complete when the kernel starts, so the tiles never wait), and consumes
// y_j = (L^T)^-1 part of block j as soon as its owner publishes it:  z_b -= L_jb^T y_j (partial sums stay in
// registers over all j), then y_b = W_b^T z_b, c_b = D y_b.  The y values themselves are the flags: the buffer is
// filled with a sentinel NaN pattern (k_scale_diag) and every consumer thread polls the 16 values it needs with
// volatile loads, so a step of the dependent chain costs one L2 round trip, two 64 x 64 matrix-vector products
// and three barriers instead of a cluster barrier and a round of global loads.  A CTA takes its place in the chain
// from a ticket drawn when it STARTS (atomicAdd on a counter zeroed by k_scale_diag), not from blockIdx: it only
// ever waits for CTAs with a smaller ticket, which are running or done already, so progress does not depend on the
// order in which the hardware dispatches the grid and needs no co-residency beyond one CTA.
constexpr int kBsStages = 4;
constexpr unsigned long long kBsSentinel = 0xFFF8DEADBEEF5AFEull;
constexpr size_t kBsSmem = (size_t)(1 + kBsStages) * NB * NB * sizeof(double) + 128;

__device__ __forceinline__ void ld_volatile_f64x2(const double *p, double &a, double &b) {
    asm volatile("ld.volatile.global.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_volatile_f64(double *p, double v) {
    asm volatile("st.volatile.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// mbarrier + bulk-copy (TMA engine) primitives: one thread arms the barrier with the byte count, the copies complete
// on it, every consumer waits on the phase parity.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// one 64 x 64 tile of the factor (tensor map over Lf as [(n+1) nbat rows][ldl columns]) as a single TMA box copy
__device__ __forceinline__ void tma_tile_g2s(void *dst, const CUtensorMap *tm, int col, int row, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::
                     "r"(smem_u32(dst)), "l"(tm), "r"(col), "r"(row), "r"(smem_u32(bar))
                 : "memory");
}

__global__ void __launch_bounds__(256)
k_chol_backsolve_lb(const __grid_constant__ CUtensorMap tmL, const double *__restrict__ Lf, const double *__restrict__ Winv,
                    const double *__restrict__ dscale, double *__restrict__ coef, double *ybuf, int n, int ldl, int nblk,
                    int nbat, int *ticket) {
    extern __shared__ double sm[];
    double *Ws = reinterpret_cast<double *>(((uintptr_t)sm + 127) & ~(uintptr_t)127);     // TMA destinations: 128-byte aligned
    double *T = Ws + NB * NB;                           // W_b [k][i]; tile ring [stage][k][col]
    __shared__ double zs[NB], red[4][NB], ysh[2][NB];
    __shared__ int s_ticket;
    const int tid = threadIdx.x, col = tid & 63, q = tid >> 6;
    if (tid == 0) s_ticket = atomicAdd(ticket, 1);
    __syncthreads();
    const int id = s_ticket, bz = id % nbat, x = id / nbat, blk = nblk - 1 - x;
    const double *L = Lf + (size_t)bz * (n + 1) * ldl;
    double *yb = ybuf + (size_t)bz * nblk * NB;
    const int i0 = blk * NB, nbk = min(NB, n - i0);
    // Staging by the TMA engine: W_b as one 32 KB bulk copy, a tile as one 64 x 64 box of the tensor map over the factor,
    // issued by one thread and completing on the stage's mbarrier (no per-thread copies or address arithmetic).
    __shared__ unsigned long long bars[kBsStages + 1];   // [stage], then W
    if (tid == 0) {
        for (int i = 0; i <= kBsStages; ++i) mbar_init(&bars[i], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 32) {
        mbar_expect_tx(&bars[kBsStages], NB * NB * sizeof(double));
        bulk_g2s(Ws, Winv + ((size_t)bz * nblk + blk) * NB * NB, NB * NB * sizeof(double), &bars[kBsStages]);
    }
    auto fetch = [&](int t) {                              // tile of block j = nblk-1-t into stage t % kBsStages
        if (t >= x || tid != 32) return;
        const int j0 = (nblk - 1 - t) * NB, st = t % kBsStages;
        mbar_expect_tx(&bars[st], NB * NB * sizeof(double));
        tma_tile_g2s(T + (size_t)st * NB * NB, &tmL, i0, bz * (n + 1) + j0, &bars[st]);
    };
#pragma unroll
    for (int t = 0; t < kBsStages - 1; ++t) fetch(t);
    if (tid < NB) zs[tid] = (tid < nbk) ? L[(size_t)n * ldl + i0 + tid] : 0.0;
    double a0 = 0.0, a1 = 0.0;
    for (int t = 0; t < x; ++t) {
        if (tid < 32) {
            // one warp polls the 64 values of block j (a hot line for every CTA below j: keep the request count low)
            const double *yj = yb + (size_t)(nblk - 1 - t) * NB + 2 * tid;
            double v0, v1;
            do {
                ld_volatile_f64x2(yj, v0, v1);
            } while ((unsigned long long)__double_as_longlong(v0) == kBsSentinel ||
                     (unsigned long long)__double_as_longlong(v1) == kBsSentinel);
            ysh[t & 1][2 * tid] = v0;
            ysh[t & 1][2 * tid + 1] = v1;
        }
        mbar_wait(&bars[t % kBsStages], (unsigned)(t / kBsStages) & 1u);      // tile t landed
        if (t == 0 && n - (nblk - 1) * NB < NB) {
            // last block: the box runs past the last unknown (rhs row, next system); those rows meet y = 0, keep them finite
            const int nv = n - (nblk - 1) * NB;
            for (int i = tid; i < (NB - nv) * NB; i += 256) T[nv * NB + i] = 0.0;
        }
        __syncthreads();        // y_j (and zero rows) visible to every thread; stage (t-1) % S and ysh[(t-1) & 1] are free again
        fetch(t + kBsStages - 1);
        const double *yv = &ysh[t & 1][16 * q];
        const double *tp = T + (size_t)(t % kBsStages) * NB * NB + (16 * q) * NB + col;
#pragma unroll
        for (int k = 0; k < 16; k += 2) {
            a0 = fma(tp[k * NB], yv[k], a0);
            a1 = fma(tp[(k + 1) * NB], yv[k + 1], a1);
        }
    }
    mbar_wait(&bars[kBsStages], 0u);                       // W landed
    red[q][col] = a0 + a1;
    __syncthreads();
    if (tid < NB) zs[tid] -= (red[0][tid] + red[1][tid]) + (red[2][tid] + red[3][tid]);
    __syncthreads();
    {
        // y_i = sum_k W[k][i] z_k  (W lower triangular, stored with its zeros)
        const double *wp = Ws + (16 * q) * NB + col;
        double y0 = 0.0, y1 = 0.0;
#pragma unroll
        for (int k = 0; k < 16; k += 2) {
            y0 = fma(wp[k * NB], zs[16 * q + k], y0);
            y1 = fma(wp[(k + 1) * NB], zs[16 * q + k + 1], y1);
        }
        __syncthreads();                                   // red (read above by tid < 64) may be rewritten
        red[q][col] = y0 + y1;
    }
    __syncthreads();
    if (tid < NB) {
        double y = (tid < nbk) ? (red[0][tid] + red[1][tid]) + (red[2][tid] + red[3][tid]) : 0.0;
        // a NaN that happens to carry the sentinel's payload (propagated from the input) must not read as "not yet
        // published" to the CTAs waiting for it
        if ((unsigned long long)__double_as_longlong(y) == kBsSentinel) y = __longlong_as_double(0x7ff8000000000000ll);
        st_volatile_f64(&yb[(size_t)blk * NB + tid], y);
        if (tid < nbk) coef[(size_t)bz * n + i0 + tid] = y * dscale[(size_t)bz * n + i0 + tid];
    }
}

}  // namespace

int solve_num_blocks(int n) { return (n + NB - 1) / NB; }

cudaError_t launch_solve(sfft_plan *p, double *d_coef) {
    const int n = p->ns, ldl = p->ldl, nbat = p->nbatch, nblk = solve_num_blocks(n);
    double *d_out = p->reduced ? p->coefr : d_coef;      // reduced solution first when the photometric ratio is constrained
    k_scale_diag<<<dim3((n + 255) / 256, nbat), 256, 0, p->stream>>>(p->M, p->dscale, p->flag, n,
                                                                    (unsigned long long *)p->ybuf, nblk * NB, kBsSentinel,
                                                                    p->flag + 2 * nbat);
    k_scale_copy<<<dim3((n + 127) / 128, (n + 1 + 15) / 16, nbat), 256, 0, p->stream>>>(p->M, p->rhs, p->dscale, p->Lf, n, ldl);
    p->launches += 2;
    cudaError_t e = cudaFuncSetAttribute(k_chol_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kStepSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_chol_update_row, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_chol_slab, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kUpdSmem);
    if (e != cudaSuccess) return e;
    for (int k = 0; k < nblk; ++k) {
        const int j1 = std::min(n, (k + 1) * NB);
        const int nslab = (n + 1 - j1 + NB - 1) / NB;                 // rows j1..n (the rhs row is row n)
        const int ntiles = k > 0 ? nslab * (nslab + 1) / 2 : 0;
        if ((long)ntiles * nbat >= 16 * 148) {
            // throughput regime: panel CTAs and the (register-lean) trailing update as two launches
            // one factoring CTA per system (it also solves slab 0), lean CTAs for the other slabs, then the update
            k_chol_step<<<dim3(1, nbat), 256, kStepSmem, p->stream>>>(p->Lf, p->Winv, p->flag, n, ldl, k, 1, 0, nblk);
            if (nslab > 1) {
                k_chol_slab<<<dim3(nslab - 1, nbat), 256, kUpdSmem, p->stream>>>(p->Lf, p->Winv, n, ldl, k, nblk);
                p->launches++;
            }
            // one CTA per segment of a tile row (operand reuse + software pipelining)
            k_chol_update_row<<<dim3(row_segments(nslab), nbat), 256, kRowSmem, p->stream>>>(p->Lf, n, ldl, k, nslab);
            p->launches += 2;
        } else {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(nslab + ntiles, nbat); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = kStepSmem;
            cfg.stream = p->stream;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
            at[0].val.programmaticStreamSerializationAllowed = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            e = cudaLaunchKernelEx(&cfg, k_chol_step, p->Lf, p->Winv, p->flag, n, ldl, k, nslab, ntiles, nblk);
            if (e != cudaSuccess) return e;
            p->launches++;
        }
    }
    e = cudaFuncSetAttribute(k_chol_backsolve_lb, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBsSmem);
    if (e != cudaSuccess) return e;
    // tensor map of the factor buffer: FP64 [(n+1) nbat rows][ldl columns], 64 x 64 boxes, zeros out of bounds
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (!fn || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
        encode = (EncodeFn)fn;
    }
    alignas(64) CUtensorMap tmL;
    const cuuint64_t gdim[2] = {(cuuint64_t)ldl, (cuuint64_t)(n + 1) * nbat}, gstr[1] = {(cuuint64_t)ldl * sizeof(double)};
    const cuuint32_t box[2] = {NB, NB}, estr[2] = {1, 1};
    if (encode(&tmL, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, p->Lf, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorInvalidValue;
    k_chol_backsolve_lb<<<dim3(nblk * nbat), 256, kBsSmem, p->stream>>>(tmL, p->Lf, p->Winv, p->dscale, d_out, p->ybuf, n, ldl,
                                                                       nblk, nbat, p->flag + 2 * nbat);
    p->launches++;
    e = cudaGetLastError();
    if (e == cudaSuccess && p->reduced) e = launch_expand_coef(p, p->coefr, d_coef);
    return e;
}

}  // namespace sfft
