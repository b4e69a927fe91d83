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
// CTA = 16 warps, one spectrum column, one barrier per step of 4 hops:
//   transform phase: warp w < 2 nseq owns the Q (w even) or P (w odd) transforms of sequence w/2, its four 8-lane
//                    groups the 4 hops; a group runs its 64-point transform in registers (radix 8 x 8) and does the
//                    one exchange IN PLACE in the 64 spectrum slots it is about to fill (skewed, conflict-free),
//                    then writes the spectrum in MMA fragment order [bin][sequence][hop];
//   MMA phase:       warp j owns bins 4j..4j+3 and keeps their ACC (Re, Im: 8 x 8 each) in registers.
// Spectra are double buffered, so warps that finish their MMAs start the next step's transforms at once; the raw
// column values are fetched two steps ahead with cp.async (by all threads: a warp keeps only a few scattered copies
// in flight); the polynomial x-weights are computed in registers.
// The packed DC/Nyquist slot (column 0 holds (X[0], X[W/2]), both real) is run as two real columns (grid.x = Nh+1).
#include "fft_regs.cuh"
#include "sfft_internal.h"

namespace sfft {
namespace {

constexpr int kOsHops = 4;                       // hops per step = K of one DMMA
constexpr int kOsBinStride = 33;                 // double2 per bin of a spectrum buffer: 8 seq x 4 hops + 1 (odd: conflict-free)
constexpr int kOsSpec = 64 * kOsBinStride;       // double2 per spectrum buffer (P or Q)
constexpr int kOsEx = 72;                        // double2 per exchange buffer of the final inverse transforms (8 x 9)
constexpr int kOsMaxImg = 4, kOsMaxXw = 3;     // images of the spectrum stack; x-weight powers u^0 .. u^2

struct OsDims { int H, Nh, nimg, nseq, L, E, Sx, HOP, RS; };

// 64-point forward DFT by a group of 8 lanes (t = lane & 7).  In: v[r] = x[t + 8 r].  Out: v[k2] = X[t + 8 k2].
// ex(i): the group's 64 exchange slots; tw[k1] = exp(-2 pi i t k1 / 64).  The slot of Y_t[k1] is skewed by k1 so
// that both the stores (lanes = t) and the loads (lanes = k1) of a quarter warp fall in eight different 16-byte banks
// whatever (odd) stride the slots have.
template <class Slot>
__device__ __forceinline__ void fft64_group(double2 (&v)[8], Slot ex, const double2 *tw, int t) {
    fft_reg<8>(v);                                            // Y_t[k1] = sum_r x[t + 8r] w8^(r k1)
#pragma unroll
    for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmulf(v[k1], tw[k1]);
#pragma unroll
    for (int k1 = 0; k1 < 8; ++k1) *ex(k1 * 8 + ((t + k1) & 7)) = v[k1];
    __syncwarp();
#pragma unroll
    for (int tt = 0; tt < 8; ++tt) v[tt] = *ex(t * 8 + ((tt + t) & 7));    // lane k1 = t gathers Y_tt[k1] w64^(tt k1)
    __syncwarp();
    fft_reg<8>(v);                                            // X[k1 + 8 k2] = sum_tt (.) w8^(tt k2)
}

// Transform phase of one step for one lane: rows t + 8r of the hop starting at staged row r0 (image row x0).
//   MODE : 0 complex column, 1 DC part (.x) and 2 Nyquist part (.y) of the packed column 0, run as real columns
//   SIDE : 0 = Q (64-row window), 1 = P (only the nkeep first rows, the rest of the window zero)
//   XP   : power of the x-weight f_i(x) = u_x^i, u_x = (2x+1)/H - 1 (exact in double for H a power of two, within an
//          ulp or two otherwise; DESIGN g8).  Computed here
//          instead of read from the plan's table: u is exact and u*u is its correctly rounded square, which is
//          what the table holds, so for H a power of two both routes weight with the very same numbers (a1).  For
//          other H the table is rounded from long double and fma(x, 2/H, 1/H - 1) can differ from it in the last
//          bit: the two routes then agree to rounding (1e-16 relative), not bit for bit.
//   P2   : H is a power of two (wrap by mask); otherwise by conditional subtraction (x0 < H + 64 for every live hop)
template <int MODE, int SIDE, int XP, bool P2>
__device__ __forceinline__ void os_transform(const double2 *rw, double2 *dst, const double2 *tw, int t, int nkeep, int x0,
                                             int H, double uscale, double uoff) {
    double2 v[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        double2 a = rw[t + 8 * r];
        if (MODE == 1) a.y = 0.0;
        if (MODE == 2) { a.x = a.y; a.y = 0.0; }
        if (XP > 0) {
            int xx = x0 + t + 8 * r;
            if (P2) xx &= H - 1;
            else { xx -= xx >= H ? H : 0; xx -= xx >= H ? H : 0; }
            const double u = fma((double)xx, uscale, uoff), w = XP == 1 ? u : u * u;
            a.x *= w;
            if (MODE == 0) a.y *= w;
        }
        if (SIDE == 1 && t + 8 * r >= nkeep) a = make_double2(0.0, 0.0);
        v[r] = a;
    }
    fft64_group(v, [dst](int i) { return dst + i * kOsBinStride; }, tw, t);
#pragma unroll
    for (int k2 = 0; k2 < 8; ++k2) dst[(t + 8 * k2) * kOsBinStride] = v[k2];
}

template <int MODE, int SIDE, bool P2>
__device__ __forceinline__ void os_transform_xp(int xp, const double2 *rw, double2 *dst, const double2 *tw, int t, int nkeep,
                                                int x0, int H, double uscale, double uoff) {
    if (xp <= 0) os_transform<MODE, SIDE, 0, P2>(rw, dst, tw, t, nkeep, x0, H, uscale, uoff);
    else if (xp == 1) os_transform<MODE, SIDE, 1, P2>(rw, dst, tw, t, nkeep, x0, H, uscale, uoff);
    else os_transform<MODE, SIDE, 2, P2>(rw, dst, tw, t, nkeep, x0, H, uscale, uoff);
}

// grid: x = column slot c (0: DC of packed column 0, Nh: its Nyquist part, else column c), y = x-range part, z = batch
template <int MODE, bool P2>
__device__ __forceinline__ void corr_os_body(const double2 *__restrict__ rhat, const Seq *__restrict__ seqs,
                                             double2 *__restrict__ G, const OsDims &d, double2 *smo) {
    double2 *SQ = smo;                                   // [2][64][33]  spectra of the 64-row windows
    double2 *SP = smo + 2 * kOsSpec;                     // [2][64][33]  spectra of the zero-padded hops (conj side)
    double2 *raw = smo + 4 * kOsSpec;                    // [2][nimg][RS] column values of the staged rows
    __shared__ double2 tw64[64];
    __shared__ Seq sseq[8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = blockIdx.x, xs = blockIdx.y, bz = blockIdx.z;
    const int col = (MODE == 2) ? 0 : c;
    const int H = d.H, HOP = d.HOP, RS = d.RS, STEP = kOsHops * d.HOP;

    if (tid < 64) {
        double s, co;
        sincospi(-(double)tid / 32.0, &s, &co);          // exp(-2 pi i tid / 64); exact at the octants
        tw64[tid] = make_double2(co, s);
    }
    if (tid < d.nseq) sseq[tid] = seqs[tid];
    // (the spectrum slots of absent sequences - slot 7 of 8 for seven sequences - are never written: whatever they
    // hold only reaches accumulator rows / columns p, q >= nseq, which are never stored)
    // this CTA's x-range: Sx parts of whole hops
    const int hops_total = (H + HOP - 1) / HOP, hpp = (hops_total + d.Sx - 1) / d.Sx;
    const int xb = min(H, xs * hpp * HOP), xe = min(H, xb + hpp * HOP);
    const int nsteps = (xe - xb + STEP - 1) / STEP;
    const double2 *rb = rhat + (size_t)bz * d.nimg * H * d.Nh + col;

    // The staged rows are fetched by all threads, one or two 16-byte items each (a warp keeps only a few scattered
    // cp.async in flight: two dedicated fetch warps took 3700 cycles per step to issue the 832 items)
    constexpr int npf = 512;
    const int img0 = tid / RS, rr0 = tid - img0 * RS;
    auto prefetch = [&](int s) {
        const int x0 = xb + s * STEP;
        double2 *rbuf = raw + (s & 1) * kOsMaxImg * RS;
        for (int img = img0, r = rr0; img < d.nimg;) {
            const int x = P2 ? ((x0 + r) & (H - 1)) : (x0 + r) % H;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(&rbuf[img * RS + r]);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(&rb[((size_t)img * H + x) * d.Nh]));
            r += npf;
            while (r >= RS) { r -= RS; ++img; }
        }
    };
    if (nsteps > 0) prefetch(0);
    if (nsteps > 1) prefetch(1);
    asm volatile("cp.async.commit_group;");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();

    // transform role: sequence, side (0: Q = 64-row window, 1: P = zero-padded hop), hop, lane of the group
    const int seq = warp >> 1, side = warp & 1, hop = lane >> 3, t = lane & 7;
    const bool live = seq < d.nseq;
    const Seq sq = live ? sseq[seq] : Seq{0, -1};
    const double uscale = 2.0 / H, uoff = 1.0 / H - 1.0;
    double2 tw[8];
#pragma unroll
    for (int k1 = 0; k1 < 8; ++k1) tw[k1] = tw64[(t * k1) & 63];
    double are[4][2], aim[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) are[i][0] = are[i][1] = aim[i][0] = aim[i][1] = 0.0;

    for (int s = 0; s < nsteps; ++s) {
        const int b = s & 1;
        if (live) {
            const int r0 = hop * HOP, x0 = xb + s * STEP + r0;
            const double2 *rw = raw + (b * kOsMaxImg + sq.img) * RS + r0;
            double2 *dst = (side ? SP : SQ) + b * kOsSpec + seq * 4 + hop;
            // the conj side keeps only the HOP rows of this hop that lie inside the CTA's x-range
            if (side) os_transform_xp<MODE, 1, P2>(sq.xw, rw, dst, tw, t, min(HOP, xe - x0), x0, H, uscale, uoff);
            else os_transform_xp<MODE, 0, P2>(sq.xw, rw, dst, tw, t, 64, x0, H, uscale, uoff);
        }
        asm volatile("cp.async.wait_group 0;" ::: "memory");      // the rows of step s+1 (fetched during step s-1) landed
        __syncthreads();                                           // spectra of step s complete; raw[b] and S[b^1] free
        if (s + 2 < nsteps) prefetch(s + 2);
        asm volatile("cp.async.commit_group;");
        const double2 *sp = SP + b * kOsSpec + (4 * warp) * kOsBinStride + lane;
        const double2 *sq2 = SQ + b * kOsSpec + (4 * warp) * kOsBinStride + lane;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double2 p = sp[i * kOsBinStride], q = sq2[i * kOsBinStride];
            dmma884(are[i], p.x, q.x);
            dmma884(are[i], p.y, q.y);
            dmma884(aim[i], p.x, q.y);
            dmma884(aim[i], -p.y, q.x);
        }
    }
    // ACC -> shared, [q*8 + p][bin] with a padded pair stride, over the spectrum buffers
    __syncthreads();
    {
        double2 *accs = smo;
        const int p = lane >> 2, q0 = 2 * (lane & 3);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            accs[(q0 * 8 + p) * 65 + 4 * warp + i] = make_double2(are[i][0], aim[i][0]);
            accs[((q0 + 1) * 8 + p) * 65 + 4 * warp + i] = make_double2(are[i][1], aim[i][1]);
        }
    }
    __syncthreads();
    // ---- inverse 64-point transform of every pair's ACC, stored at the lags rho < L:  G = conj(FFT(conj ACC)) / 64 ----
    {
        const int g = tid >> 3, q = g >> 3, p = g & 7;
        double2 *ex2 = smo + 64 * 65 + g * kOsEx;          // past the ACC copy (runs on into the raw staging area)
        double2 v[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) { const double2 a = smo[g * 65 + t + 8 * r]; v[r] = make_double2(a.x, -a.y); }
        fft64_group(v, [ex2](int i) { return ex2 + i + (i >> 3); }, tw, t);
        if (p < d.nseq && q < d.nseq) {
            double2 *Gm = G + (((size_t)bz * d.Sx + xs) * (d.Nh + 1) + c) * d.E + (size_t)(p * d.nseq + q) * d.L;
#pragma unroll
            for (int k2 = 0; k2 < 8; ++k2) {
                const int rho = t + 8 * k2;
                if (rho < d.L) Gm[rho] = make_double2(v[k2].x * (1.0 / 64.0), MODE ? 0.0 : -v[k2].y * (1.0 / 64.0));
            }
        }
    }
}

template <bool P2>
__global__ void __launch_bounds__(512, 1)
k_corr_os(const double2 *__restrict__ rhat, const Seq *__restrict__ seqs, double2 *__restrict__ G, OsDims d) {
    extern __shared__ double2 smo[];
    const int c = blockIdx.x;                            // uniform per CTA
    if (c == 0) corr_os_body<1, P2>(rhat, seqs, G, d, smo);
    else if (c == d.Nh) corr_os_body<2, P2>(rhat, seqs, G, d, smo);
    else corr_os_body<0, P2>(rhat, seqs, G, d, smo);
}

size_t corr_os_smem(const OsDims &d) {
    const size_t main_loop = (size_t)(4 * kOsSpec + 2 * kOsMaxImg * d.RS) * sizeof(double2);
    const size_t epilogue = (size_t)(64 * 65 + 64 * kOsEx) * sizeof(double2);      // ACC copy + 64 exchange buffers
    return main_loop > epilogue ? main_loop : epilogue;
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
    OsDims d{p->H, p->Nh, p->nimg, p->nseq, p->L, p->E, p->Sx, corr_os_hop(p), 0};
    d.RS = (kOsHops - 1) * d.HOP + 64;
    const size_t smem = corr_os_smem(d);
    const bool p2 = (p->H & (p->H - 1)) == 0;
    cudaError_t e = cudaFuncSetAttribute(p2 ? k_corr_os<true> : k_corr_os<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(p->Nh + 1, p->Sx, p->nbatch);
    if (p2) k_corr_os<true><<<grid, 512, smem, p->stream>>>(p->rhat, p->dt.seqs, p->G, d);
    else k_corr_os<false><<<grid, 512, smem, p->stream>>>(p->rhat, p->dt.seqs, p->G, d);
    p->launches++;
    return cudaGetLastError();
}

}  // namespace sfft

