// Steps a3+a4 (x-direction): cross-spectra and the "saccadic" restriction to the kernel lags,
// on the FP64 tensor cores.
//
// After the row transform (rowfft.cu) every correlation array of App. B
// factorises over the spectrum columns m:
//   Omega_{tb,t}(rho,eps) = sum_{x,y} R^tb(x,y) R^t(x+rho,y+eps)                              (B6, DESIGN g2)
//     = (1/W) sum_m w_m Re[ G_{tb,t}(rho; m) exp(+2 pi i m eps / W) ],   w_0 = w_{W/2} = 1, else 2
//   G_{p,q}(rho; m) = sum_x conj(z_p(x,m)) z_q((x+rho) mod H, m),        z_t(x,m) = f_i(x) r_j(x,m)
// and likewise Theta (q = S, B14).  The normal matrix reads Omega only at |rho| <= L-1 and Theta at
// |rho| <= w (B5-B15), so the x-direction is evaluated at those lags only: the paper's full-size
// correlation arrays (and the column transforms that would produce them) are never formed.
// Negative lags come from  G_{p,q}(-rho) = conj(G_{q,p}(rho)),  so only rho = 0..L-1 is computed,
// for all ordered pairs.
//
// For one column m this is a small dense contraction over x with a Hankel right operand:
//   rows    : Re z_p, Im z_p of four sequences p                       (8 real rows)
//   columns : z_q(x + rho) for eight consecutive lags rho              (8 columns, Re and Im apart)
// i.e. two mma.sync.m8n8k4.f64 (DMMA) per 4 x-values give 4 x 8 complex lag sums with no wasted
// multiply:  Re G = Cr[p] + Ci[p+4],  Im G = Ci[p] - Cr[p+4]   (Cr = A Br, Ci = A Bi).
// The Hankel operand needs no data movement: lane (k, n) of the B fragment reads z_q(x0 + k + n + rho0)
// straight from the x-contiguous shared-memory plane.  When L-1 is a multiple of 8 lag 0 uses one extra
// block whose columns are eight N-side sequences at rho = 0 (blocks then start at lag 1); otherwise the
// blocks start at lag 0.  Each job carries its own block list (only the lags the normal system reads:
// L-1 between kernel terms, w against S, none for S with S) and its own x-ranges (compactly supported
// B-spline x-factors: outside the overlap of the two supports every product vanishes identically).  The packed DC/Nyquist slot (column 0 holds (X[0], X[W/2]), both
// real) falls out of the same arithmetic: Cr[p] is the DC sum and Ci[p+4] the Nyquist sum.
//
// CTA = 8 warps = 2 columns x 2 row blocks x 2 halves of the block list; two CTAs per SM overlap one
// CTA's staging with the other's MMAs.  FP64-MMA bound.
#include "sfft_internal.h"

namespace sfft {
namespace {

__device__ __forceinline__ double lds_f64(unsigned addr) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
    return v;
}

// MMAs of one staged tile for a warp with exactly NB blocks (compile-time trip counts, no predication:
// mma.sync under a predicate costs a warp re-convergence per instruction).
template <int NB, int XS>
__device__ __forceinline__ void corr_tile_mma(double (&acc)[kCorrBlk][2][2], unsigned aA, const unsigned (&aB)[kCorrBlk],
                                              int kmax) {
#pragma unroll 2
    for (int kk = 0; kk < kmax; kk += 4) {
        const double a = lds_f64(aA + kk * 8);
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int pt = 0; pt < 2; ++pt) dmma884(acc[i][pt], a, lds_f64(aB[i] + (pt * 2 * XS + kk) * 8));
    }
}

template <int XT, int NLB>
struct CorrCfg {
    static constexpr int ROWS = XT + 8 * NLB;              // staged x-rows per tile (largest lag offset + fragment extent)
    static constexpr int XS = ((ROWS + 7) / 16) * 16 + 8;  // plane stride, = 8 mod 16 (conflict-free staging stores)
    static constexpr int SS = 4 * XS + 4;                  // slot stride [part 2][col 2][XS] + 4 (conflict-free A loads)
    // operand planes + the raw cp.async staging buffers of one tile (value 16 bytes + x-weight 8 bytes per item)
    static constexpr size_t SMEM = (size_t)kCorrSlots * SS * sizeof(double) + (size_t)kCorrSlots * ROWS * kCorrCols * (sizeof(double2) + sizeof(double));
};

// grid: x = column pair, y = job * Sx + xs, z = batch.  block: 256.
template <int XT, int NLB>
__global__ void __launch_bounds__(256, 2)
k_corr_mma(const double2 *__restrict__ rhat, const double *__restrict__ xwt, const Seq *__restrict__ seqs,
           const CorrJob *__restrict__ jobs, double2 *__restrict__ G, int H, int Nh, int nimg, int nseq, int L, int E,
           int Sx) {
    using C = CorrCfg<XT, NLB>;
    constexpr int ROWS = C::ROWS, XS = C::XS, SS = C::SS;
    extern __shared__ double sm[];
    __shared__ CorrJob job;
    __shared__ Seq sseq[kCorrSlots];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int col = warp & 1, mb = (warp >> 1) & 1, nh = warp >> 2;
    const int jb = blockIdx.y / Sx, xs = blockIdx.y - jb * Sx, bz = blockIdx.z;
    const int m0 = blockIdx.x * kCorrCols;

    if (tid < (int)(sizeof(CorrJob) / sizeof(int))) reinterpret_cast<int *>(&job)[tid] = reinterpret_cast<const int *>(&jobs[jb])[tid];
    // only the zero plane has to be cleared: every staged plane is rewritten in full (rows < ROWS) for each tile
    for (int i = tid; i < SS; i += 256) sm[kCorrZero * SS + i] = 0.0;
    __syncthreads();
    if (tid < job.nstage) sseq[tid] = seqs[job.stage_seq[tid]];

    const double2 *rhat_b = rhat + (size_t)bz * nimg * H * Nh;
    const int row = lane >> 2, kq = lane & 3;
    // per-lane fragment bases (doubles): A = rows (Re, Im) of four M-side sequences; B = per block, a Hankel read
    // of one plane at its first lag, or (lag-0 block) one plane per column
    const unsigned sm0 = (unsigned)__cvta_generic_to_shared(sm);
    const unsigned aA = sm0 + 8u * (job.mslot[mb][row & 3] * SS + ((row >> 2) * 2 + col) * XS + kq);
    const int nb = job.nblk[nh];
    unsigned aB[kCorrBlk];
#pragma unroll
    for (int i = 0; i < kCorrBlk; ++i) {
        const int sl = job.blk_slot[nh][i];
        aB[i] = sm0 + 8u * ((sl >= 0 ? sl * SS + job.blk_lag[nh][i] + row : job.zslot[row] * SS) + col * XS + kq);
    }

    double acc[kCorrBlk][2][2];
#pragma unroll
    for (int i = 0; i < kCorrBlk; ++i)
#pragma unroll
        for (int pt = 0; pt < 2; ++pt) acc[i][pt][0] = acc[i][pt][1] = 0.0;

    const int nitems = job.nstage * ROWS * kCorrCols;
    // this CTA's part of each x-range: Sx parts of whole 4-row steps
    int pb0, pe0, pb1 = 0, pe1 = 0;
    {
        const int rb = job.xbeg[0], re = job.xend[0], plen = (((re - rb) / 4 + Sx - 1) / Sx) * 4;
        pb0 = rb + xs * plen; pe0 = min(re, pb0 + plen);
        if (job.nrange > 1) {
            const int rb1 = job.xbeg[1], re1 = job.xend[1], plen1 = (((re1 - rb1) / 4 + Sx - 1) / Sx) * 4;
            pb1 = rb1 + xs * plen1; pe1 = min(re1, pb1 + plen1);
        }
    }
    // tile cursor (range, first row); range 2 = done
    auto settle = [&](int &r, int &x) {
        if (r == 0 && x >= pe0) { r = 1; x = pb1; }
        if (r == 1 && x >= pe1) r = 2;
    };
    // The raw spectrum values of a tile are fetched with cp.async into a staging buffer while the MMAs of the
    // previous tile run (no registers held across the MMA phase); each thread later converts the items it
    // fetched itself (weight, Re/Im split) into the operand planes.
    double2 *raw = reinterpret_cast<double2 *>(sm + kCorrSlots * SS);
    double *raww = reinterpret_cast<double *>(raw + kCorrSlots * ROWS * kCorrCols);      // x-weight of every item
    auto prefetch = [&](int x0) {
        for (int i = tid; i < nitems; i += 256) {
            const int c = i & 1, r = (i >> 1) % ROWS, si = (i >> 1) / ROWS;
            const int x = (x0 + r) & (H - 1);
            const Seq sq = sseq[si];
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&raw[i]);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst),
                         "l"(&rhat_b[((size_t)sq.img * H + x) * Nh + m0 + c]));
            if (sq.xw >= 0) {
                const unsigned dw = (unsigned)__cvta_generic_to_shared(&raww[i]);
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dw), "l"(&xwt[(size_t)sq.xw * H + x]));
            }
        }
        asm volatile("cp.async.commit_group;");
    };
    int crg = 0, cx = pb0;
    settle(crg, cx);
    __syncthreads();                    // sseq visible
    if (crg < 2) prefetch(cx);
    while (crg < 2) {
        int nrg = crg, nx = cx + XT;
        settle(nrg, nx);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();                // every warp is done with the planes of the previous tile
        // ---- stage the tile: weighted sequences, split into Re / Im planes, x-contiguous ----
        for (int i = tid; i < nitems; i += 256) {
            const int c = i & 1, r = (i >> 1) % ROWS, si = (i >> 1) / ROWS;
            const Seq sq = sseq[si];
            double2 v = raw[i];
            if (sq.xw >= 0) { const double wgt = raww[i]; v.x *= wgt; v.y *= wgt; }
            double *pl = sm + job.stage_slot[si] * SS + c * XS + r;
            pl[0] = v.x;
            pl[2 * XS] = v.y;
        }
        if (nrg < 2) prefetch(nx);      // own slots of the raw buffer only: no barrier needed before reuse
        __syncthreads();
        // ---- MMAs ----
        const int kmax = min(XT, (crg == 0 ? pe0 : pe1) - cx);
        switch (nb) {               // warp-uniform
            case 1: corr_tile_mma<1, XS>(acc, aA, aB, kmax); break;
            case 2: corr_tile_mma<2, XS>(acc, aA, aB, kmax); break;
            case 3: corr_tile_mma<3, XS>(acc, aA, aB, kmax); break;
            case 4: corr_tile_mma<4, XS>(acc, aA, aB, kmax); break;
            case 5: corr_tile_mma<5, XS>(acc, aA, aB, kmax); break;
            case 6: corr_tile_mma<6, XS>(acc, aA, aB, kmax); break;
            case 7: corr_tile_mma<7, XS>(acc, aA, aB, kmax); break;
            case 8: corr_tile_mma<8, XS>(acc, aA, aB, kmax); break;
            default: break;
        }
        crg = nrg; cx = nx;
    }

    // ---- epilogue: combine the Re/Im row halves and store G[b][xs][m][e] ----
    const int mcol = m0 + col;
    double2 *Gm = G + (((size_t)bz * Sx + xs) * (Nh + 1) + mcol) * E;
    double2 *Gn = G + (((size_t)bz * Sx + xs) * (Nh + 1) + Nh) * E;     // Nyquist row (used by column 0 only)
    const int p = job.mseq[mb][row & 3];
#pragma unroll
    for (int i = 0; i < kCorrBlk; ++i) {
        if (i >= nb) continue;
        const int sl = job.blk_slot[nh][i];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double cr = acc[i][0][q], ci = acc[i][1][q];
            const double ocr = __shfl_xor_sync(0xffffffffu, cr, 16), oci = __shfl_xor_sync(0xffffffffu, ci, 16);
            if (row >= 4) continue;
            const int nn = 2 * kq + q;
            int rho, qs;
            if (sl < 0) { rho = 0; qs = job.zseq[nn]; }
            else { rho = job.blk_lag[nh][i] + nn; qs = nn < job.blk_nlag[nh][i] ? job.blk_seq[nh][i] : -1; }
            if (p < 0 || qs < 0 || rho >= L) continue;
            const int e = (p * nseq + qs) * L + rho;
            if (mcol == 0) {
                Gm[e] = make_double2(cr, 0.0);
                Gn[e] = make_double2(oci, 0.0);
            } else {
                Gm[e] = make_double2(cr + oci, ci - ocr);
            }
        }
    }
}

template <int XT, int NLB>
cudaError_t launch_t(sfft_plan *p) {
    using C = CorrCfg<XT, NLB>;
    auto kern = k_corr_mma<XT, NLB>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    dim3 grid(p->Nh / kCorrCols, (unsigned)p->jobs.size() * p->Sx, p->nbatch);
    kern<<<grid, 256, C::SMEM, p->stream>>>(p->rhat, p->dt.xwt, p->dt.seqs, p->dt.jobs, p->G, p->H, p->Nh, p->nimg,
                                            p->nseq, p->L, p->E, p->Sx);
    p->launches++;
    return cudaGetLastError();
}

template <int XT>
cudaError_t launch_x(sfft_plan *p) {
    switch (p->nlb) {
        case 0: return launch_t<XT, 0>(p);
        case 1: return launch_t<XT, 1>(p);
        case 2: return launch_t<XT, 2>(p);
        case 3: return launch_t<XT, 3>(p);
        case 4: return launch_t<XT, 4>(p);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_corr(sfft_plan *p) {
    if (corr_use_os(p)) return launch_corr_os(p);
    return (p->H / p->Sx) >= 64 ? launch_x<64>(p) : launch_x<32>(p);
}

}  // namespace sfft
