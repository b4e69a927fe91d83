// Steps a3+a4 (x-direction), sectioned form: cross-spectra and the "saccadic" restriction to the kernel lags by
// overlap-save correlation with 64-point FFTs along x.  Used when the model has at most 8 column sequences
// (polynomial bases up to DK = 2: 6 kernel terms + S); corr.cu keeps the direct tensor-core lag sums for the
// many-term / compactly supported (B-spline) bases.
//
// Per spectrum column m the normal system needs (corr.cu; App. B; B6, B14 with DESIGN g2)
//   G_{p,q}(rho; m) = sum_x conj(z_p(x,m)) z_q((x+rho) mod H, m),   0 <= rho <= L-1,   z_t(x,m) = f_i(x) r_j(x,m),
// for all ordered pairs of the nseq sequences.  The paper obtains the full-length correlation from full-size DFTs
// and reads it at the lags; only rho < L is ever read, so the x axis is cut in hops of HOP = 64 - (L-1) rows:
//   P_p = FFT64(z_p[x0 .. x0+HOP) zero-padded),   Q_q = FFT64(z_q[x0 .. x0+64) wrapped mod H),
//   ACC_{p,q}[k] += conj(P_p[k]) Q_q[k]   over all hops,
//   G_{p,q}(rho) = (1/64) sum_k ACC_{p,q}[k] exp(+2 pi i k rho / 64),   exact for rho <= 64 - HOP (n + rho <= 63 never wraps).
// Cost per hop and column: 2 nseq FFT64 + 64 bins x (nseq x nseq complex MAC): ~9 GFLOP at config 4 against the
// 60 GFLOP the direct lag sums execute.
//
// The accumulation over hops is, per frequency bin, a rank-(number of hops) update of an 8 x 8 complex matrix:
// a dense contraction with K = hops, run on the FP64 tensor cores (mma.sync.m8n8k4.f64, K = 4 hops per step):
//   Re ACC += Pr^T Qr + Pi^T Qi,   Im ACC += Pr^T Qi - Pi^T Qr        (4 DMMA per bin per 4 hops).
//
// CTA = 16 warps, one spectrum column, warp specialised:
//   warps 0..7  (producers): warp s owns sequence s, its four 8-lane groups own the 4 hops of a step; each group
//               runs the P and Q transforms of its (sequence, hop) in registers (radix 8 x 8, one padded
//               shared-memory exchange) and writes the spectra in MMA fragment order [bin][sequence][hop];
//   warps 8..15 (consumers): warp j owns bins 8j..8j+7 and keeps their ACC (Re, Im: 8 x 8 each) in registers;
//   two spectrum buffers, named barriers full[2] / empty[2]; the raw column values and x-weights of the next step
//   are fetched with cp.async while the current one is transformed.
// The packed DC/Nyquist slot (column 0 holds (X[0], X[W/2]), both real) is run as two real columns (grid.x = Nh+1).
#include "fft_regs.cuh"
#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int kOsHops = 4;                       // hops per step = K of one DMMA
constexpr int kOsBinStride = 36;                 // double2 per bin of a spectrum buffer: 8 seq x 4 hops + 4 pad
constexpr int kOsSpec = 64 * kOsBinStride;       // double2 per spectrum buffer (P or Q)
constexpr int kOsEx = 72;                        // double2 per FFT group exchange buffer (8 x 9, padded)
constexpr int kOsMaxImg = 4, kOsMaxXw = 3;

struct OsDims { int H, Nh, nimg, nKa, nseq, L, E, Sx, HOP, RS; };

__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) {
    __threadfence_block();
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}

// 64-point forward DFT by a group of 8 lanes (t = lane & 7).  In: v[r] = x[t + 8 r].  Out: v[k2] = X[t + 8 k2].
// ex: the group's exchange buffer (kOsEx entries); tw[k1] = exp(-2 pi i t k1 / 64).
__device__ __forceinline__ void fft64_group(double2 (&v)[8], double2 *ex, const double2 *tw, int t) {
    fft_reg<8>(v);                                            // Y_t[k1] = sum_r x[t + 8r] w8^(r k1)
#pragma unroll
    for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmulf(v[k1], tw[k1]);
#pragma unroll
    for (int k1 = 0; k1 < 8; ++k1) ex[t * 9 + k1] = v[k1];
    __syncwarp();
#pragma unroll
    for (int tt = 0; tt < 8; ++tt) v[tt] = ex[tt * 9 + t];    // lane k1 = t gathers Y_tt[k1] w64^(tt k1)
    __syncwarp();
    fft_reg<8>(v);                                            // X[k1 + 8 k2] = sum_tt (.) w8^(tt k2)
}

// grid: x = column slot c (0: DC of packed column 0, Nh: its Nyquist part, else column c), y = x-range part, z = batch
__global__ void __launch_bounds__(512, 1)
k_corr_os(const double2 *__restrict__ rhat, const double *__restrict__ xwt, const Seq *__restrict__ seqs,
          double2 *__restrict__ G, OsDims d) {
    extern __shared__ double2 smo[];
    double2 *SP = smo;                                   // [2][64][36]  spectra of the zero-padded hops (conj side)
    double2 *SQ = smo + 2 * kOsSpec;                     // [2][64][36]  spectra of the 64-row windows
    double2 *raw = smo + 4 * kOsSpec;                    // [2][nimg][RS] column values of the staged rows
    double2 *exb = raw + 2 * kOsMaxImg * d.RS;           // [8 warps][4 groups][72]
    double *wts = reinterpret_cast<double *>(exb + 8 * 4 * kOsEx);   // [2][nKa][RS] x-weights of the staged rows
    __shared__ double2 tw64[64];
    __shared__ Seq sseq[8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x, xs = blockIdx.y, bz = blockIdx.z;
    const int mode = (c == 0) ? 1 : (c == d.Nh ? 2 : 0), col = (c == d.Nh) ? 0 : c;
    const int H = d.H, HOP = d.HOP, RS = d.RS, STEP = kOsHops * d.HOP;

    if (tid < 64) {
        double s, co;
        sincospi(-(double)tid / 32.0, &s, &co);          // exp(-2 pi i tid / 64); exact at the octants
        tw64[tid] = make_double2(co, s);
    }
    if (tid < d.nseq) sseq[tid] = seqs[tid];
    for (int i = tid; i < 4 * kOsSpec; i += 512) smo[i] = make_double2(0.0, 0.0);
    // this CTA's x-range: Sx parts of whole hops
    const int hops_total = (H + HOP - 1) / HOP, hpp = (hops_total + d.Sx - 1) / d.Sx;
    const int xb = min(H, xs * hpp * HOP), xe = min(H, xb + hpp * HOP);
    const int nsteps = (xe - xb + STEP - 1) / STEP;
    const double2 *rb = rhat + (size_t)bz * d.nimg * H * d.Nh + col;
    __syncthreads();

    if (warp < 8) {
        // ------------------------------------------------ producers ------------------------------------------------
        const int hop = lane >> 3, t = lane & 7, seq = warp;
        double2 *ex = exb + (warp * 4 + hop) * kOsEx;
        const bool live = seq < d.nseq;
        const Seq sq = live ? sseq[seq] : Seq{0, -1};
        double2 tw[8];
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) tw[k1] = tw64[(t * k1) & 63];
        auto prefetch = [&](int s) {
            const int x0 = xb + s * STEP, b = s & 1;
            for (int i = tid; i < d.nimg * RS; i += 256) {
                const int img = i / RS, r = i - img * RS, x = (x0 + r) & (H - 1);
                const unsigned dst = (unsigned)__cvta_generic_to_shared(&raw[(b * kOsMaxImg + img) * RS + r]);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(&rb[((size_t)img * H + x) * d.Nh]));
            }
            for (int i = tid; i < d.nKa * RS; i += 256) {
                const int f = i / RS, r = i - f * RS, x = (x0 + r) & (H - 1);
                const unsigned dst = (unsigned)__cvta_generic_to_shared(&wts[(b * kOsMaxXw + f) * RS + r]);
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(&xwt[(size_t)f * H + x]));
            }
            asm volatile("cp.async.commit_group;");
        };
        if (nsteps > 0) prefetch(0);
        for (int s = 0; s < nsteps; ++s) {
            const int b = s & 1;
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            bar_sync(5, 256);                              // raw[b] of every producer thread landed; step s-1 fully read
            if (s + 1 < nsteps) prefetch(s + 1);
            if (s >= 2) bar_sync(3 + b, 512);              // empty[b]: the consumers are done with the spectra of step s-2
            if (live) {
                const int r0 = hop * HOP;
                const double2 *rw = raw + (b * kOsMaxImg + sq.img) * RS + r0;
                const double *wt = wts + (b * kOsMaxXw + (sq.xw >= 0 ? sq.xw : 0)) * RS + r0;
                double2 v[8], q[8];
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    double2 a = rw[t + 8 * r];
                    if (mode == 1) a.y = 0.0;
                    else if (mode == 2) { a.x = a.y; a.y = 0.0; }
                    if (sq.xw >= 0) { const double w = wt[t + 8 * r]; a.x *= w; a.y *= w; }
                    q[r] = a;
                    // the conj side keeps only the HOP rows of this hop that lie inside the CTA's x-range
                    const bool keep = (t + 8 * r < HOP) && (xb + s * STEP + r0 + t + 8 * r < xe);
                    v[r] = keep ? a : make_double2(0.0, 0.0);
                }
                fft64_group(q, ex, tw, t);
                double2 *dq = SQ + b * kOsSpec + seq * 4 + hop;
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) dq[(t + 8 * k2) * kOsBinStride] = q[k2];
                fft64_group(v, ex, tw, t);
                double2 *dp = SP + b * kOsSpec + seq * 4 + hop;
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) dp[(t + 8 * k2) * kOsBinStride] = v[k2];
            }
            bar_arrive(1 + b, 512);                        // full[b]
        }
    } else {
        // ------------------------------------------------ consumers ------------------------------------------------
        const int j = warp - 8;
        double are[8][2], aim[8][2];
#pragma unroll
        for (int i = 0; i < 8; ++i) are[i][0] = are[i][1] = aim[i][0] = aim[i][1] = 0.0;
        for (int s = 0; s < nsteps; ++s) {
            const int b = s & 1;
            bar_sync(1 + b, 512);                          // full[b]
            const double2 *sp = SP + b * kOsSpec + (8 * j) * kOsBinStride + lane;
            const double2 *sq2 = SQ + b * kOsSpec + (8 * j) * kOsBinStride + lane;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const double2 p = sp[i * kOsBinStride], q = sq2[i * kOsBinStride];
                dmma884(are[i], p.x, q.x);
                dmma884(are[i], p.y, q.y);
                dmma884(aim[i], p.x, q.y);
                dmma884(aim[i], -p.y, q.x);
            }
            if (s + 2 < nsteps) bar_arrive(3 + b, 512);    // empty[b]
        }
        // ACC -> shared, [q*8 + p][bin] with a padded pair stride, over the spectrum buffers: the producers wrote
        // them for the last time before the last full[] barrier; every consumer must have read its last operands
        bar_sync(6, 256);
        double2 *accs = smo;
        const int p = lane >> 2, q0 = 2 * (lane & 3);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            accs[(q0 * 8 + p) * 65 + 8 * j + i] = make_double2(are[i][0], aim[i][0]);
            accs[((q0 + 1) * 8 + p) * 65 + 8 * j + i] = make_double2(are[i][1], aim[i][1]);
        }
    }
    __syncthreads();
    // ---- inverse 64-point transform of every pair's ACC, stored at the lags rho < L:  G = conj(FFT(conj ACC)) / 64 ----
    {
        const int g = tid >> 3, t = tid & 7, q = g >> 3, p = g & 7;
        double2 *ex2 = smo + 64 * 65 + g * kOsEx;
        double2 tw[8];
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) tw[k1] = tw64[(t * k1) & 63];
        double2 v[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) { const double2 a = smo[g * 65 + t + 8 * r]; v[r] = make_double2(a.x, -a.y); }
        fft64_group(v, ex2, tw, t);
        if (p < d.nseq && q < d.nseq) {
            double2 *Gm = G + (((size_t)bz * d.Sx + xs) * (d.Nh + 1) + c) * d.E + (size_t)(p * d.nseq + q) * d.L;
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int rho = t + 8 * k2;
                if (rho < d.L) Gm[rho] = make_double2(v[k2].x * (1.0 / 64.0), mode ? 0.0 : -v[k2].y * (1.0 / 64.0));
            }
        }
    }
}

size_t corr_os_smem(const OsDims &d) {
    return (size_t)(4 * kOsSpec + 2 * kOsMaxImg * d.RS + 8 * 4 * kOsEx) * sizeof(double2) + (size_t)2 * kOsMaxXw * d.RS * sizeof(double);
}

}  // namespace

// The sectioned kernel serves dense (polynomial) bases with at most 8 column sequences.
bool corr_os_possible(const sfft_plan *p) {
    return p->basis == SFFT_BASIS_POLY && p->nseq <= 8 && p->nimg <= kOsMaxImg && p->nKa <= kOsMaxXw && p->L <= 33;
}
bool corr_use_os(const sfft_plan *p) { return p->corr_route != 1 && corr_os_possible(p); }

int corr_os_hop(const sfft_plan *p) { return 64 - (p->L - 1); }

// x-range parts: whole waves of one CTA per SM; a part pays ~2 steps of prologue/epilogue
int corr_os_split(const sfft_plan *p) {
    const int HOP = corr_os_hop(p), hops = (p->H + HOP - 1) / HOP;
    int best_sx = 1;
    double best = 1e300;
    for (int sx = 1; sx <= 8; sx *= 2) {
        const int hpp = (hops + sx - 1) / sx;
        if (sx > 1 && hpp < kOsHops) break;
        const double ctas = (double)(p->Nh + 1) * sx * p->nbatch;
        const double cost = ceil(ctas / 148.0) * ((hpp + kOsHops - 1) / kOsHops + 2.0);
        if (cost < best) { best = cost; best_sx = sx; }
    }
    return best_sx;
}

cudaError_t launch_corr_os(sfft_plan *p) {
    OsDims d{p->H, p->Nh, p->nimg, p->nKa, p->nseq, p->L, p->E, p->Sx, corr_os_hop(p), 0};
    d.RS = (kOsHops - 1) * d.HOP + 64;
    const size_t smem = corr_os_smem(d);
    cudaError_t e = cudaFuncSetAttribute(k_corr_os, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(p->Nh + 1, p->Sx, p->nbatch);
    k_corr_os<<<grid, 512, smem, p->stream>>>(p->rhat, p->dt.xwt, p->dt.seqs, p->G, d);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft
