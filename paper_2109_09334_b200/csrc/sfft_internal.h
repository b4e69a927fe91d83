// Internal declarations of libsfft_b200 (not part of the C ABI; see include/sfft.h).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/sfft.h"

namespace sfft {

#ifdef __CUDACC__
// v mod N (any sign); mask = N - 1 when N is a power of two, else < 0
__device__ __forceinline__ int wrap_index(int v, int N, int mask) {
    if (mask >= 0) return v & mask;
    v %= N;
    return v < 0 ? v + N : v;
}
// One FP64 tensor-core MMA (DMMA on sm_100a): C[8x8] += A[8x4] B[4x8].  Fragments: a = A[lane>>2][lane&3],
// b = B[lane&3][lane>>2], c[q] = C[lane>>2][2*(lane&3) + q].
__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c[0]), "+d"(c[1])
        : "d"(a), "d"(b));
}
#endif

constexpr int kProfMarks = 12;     // event marks per profiled step (see sfft_plan_profile_read)
constexpr int kCorrCols = 2;       // spectrum columns (m) per CTA of the correlation kernel
constexpr int kCorrNSlots = 8;     // N-side (shifted) sequence planes per correlation job: slots 0..7
constexpr int kCorrZero = 8;       // slot of the all-zero plane (absent M-side rows, absent lag-0 columns)
constexpr int kCorrSlots = 17;     // shared-memory sequence planes per CTA: 0..7 N side, 8 zero, 9..16 extra M side
constexpr int kCorrBlk = 8;        // N-side 8-lag blocks per warp half (16 per job)
constexpr int kLagChunk = 32;      // spectrum columns per partial sum of the y-direction inverse DFT

// One column-sequence of the x-direction correlation:  z_s(x, m) = xw[x] * rhat[img][x][m]
//   img : row-transformed image of the spectrum stack (0..nKa-1: g_j(y) R, nKa: S)
//   xw  : row of the x-weight table (kernel x-basis function f_i), < 0 = no weight
struct Seq { int img; int xw; };

// One job of k_corr_mma: ordered pairs (p in mseq) x (q on the N side) at the lags its blocks list,
//   G_{p,q}(rho; m) = sum_x conj(z_p(x,m)) z_q((x+rho) mod H, m),   x over the job's x-ranges.
// An N-side block is either eight consecutive lags of ONE sequence (Hankel operand read in place) or the
// lag-0 block, whose eight columns are eight different sequences at rho = 0.
struct CorrJob {
    int mseq[2][4];         // M-side sequence ids of the two 4-row blocks; -1 = none
    int mslot[2][4];        // their plane slots (kCorrZero if none)
    int nstage;             // number of staged planes
    int stage_slot[kCorrSlots], stage_seq[kCorrSlots];
    int nblk[2];            // blocks of each warp half
    int blk_slot[2][kCorrBlk];   // plane slot of the block's sequence; -1 = the lag-0 block
    int blk_seq[2][kCorrBlk];    // its sequence id
    int blk_lag[2][kCorrBlk];    // first lag of the block
    int blk_nlag[2][kCorrBlk];   // valid lags (1..8)
    int zslot[8], zseq[8];  // lag-0 block: plane slot (kCorrZero if none) and sequence id (-1) of each column
    int nrange;             // x-ranges (1 or 2; bounds are multiples of 4); outside them every product vanishes
    int xbeg[2], xend[2];
};

// One row of a lag table produced by the y-direction pruned inverse DFT:
//   dst[eps + hw] = (1/W) sum_m w_m Re[ G[e][m] exp(+2 pi i m (sgn*eps) / W) ],  |eps| <= hw
struct LagUnit { int e; int sgn; int hw; int dst_off; };

struct DeviceTables {
    double *xwt = nullptr;      // [nKa + nBa][H]   x-axis basis tables (kernel rows first)
    double *gK = nullptr;       // [nKa][W]         kernel y-axis basis
    double *gB = nullptr;       // [nBa][W]         background y-axis basis
    double2 *twW = nullptr;     // [W]              exp(-2 pi i k / W)
    double2 *twM = nullptr;     // [2 M]            exp(-2 pi i k / (2M)): twiddles of the M-point transforms of the chirp-z row DFT (W not a power of two)
    double2 *chirp = nullptr;   // [W/2]            exp(-i pi n^2 / (W/2))
    double2 *bhat = nullptr;    // [M]              M-point DFT of the wrapped conjugate chirp
    double2 *lagtw = nullptr;   // [Nh+1][L]        (w_m cos, w_m sin)(2 pi m k / W) / W
    double *cq = nullptr;       // [NC][nMom]       POLY: Q_c = sum_a cq[c][a] mu_a + border terms (binomial shift of g'_j by beta)
    double *cwr = nullptr;      // [NC][w]          POLY: coefficients of the |beta| row pixels whose shifted partner wraps
    double *cy = nullptr;       // [NC][W]          g_jb(y) g'_j((y+beta) mod W),  c = (jb*nBa + j)*L + beta+w
    double *fx = nullptr;       // [NC][H]          f_ib(x) f'_i((x+alpha) mod H), c = (ib*nBa + i)*L + alpha+w
    double *phi0 = nullptr;     // [FB][FB]         M_bb (plan constant)
    Seq *seqs = nullptr;
    CorrJob *jobs = nullptr;
    LagUnit *units = nullptr;
    int *kti = nullptr, *ktj = nullptr, *bti = nullptr, *btj = nullptr;
    int *kdec = nullptr;        // [FK*L*L]         t << 16 | (alpha+w) << 8 | (beta+w) of every kernel unknown (gather.cu)
    int *ridx = nullptr;        // [ns]             full-layout index of every solved unknown (reduced systems: cpr, rectangular kernels)
    int *fmap = nullptr;        // [n]              solved index of every full-layout unknown, -1 = fixed at zero
};

}  // namespace sfft

struct sfft_plan {
    int H = 0, W = 0, L = 0, w = 0, DK = 0, DB = 0, basis = 0, nbatch = 1;
    int FK = 0, FB = 0, nKa = 0, nBa = 0, n = 0, Nh = 0;
    bool corr_os = false; int os_hop = 0;   // the build takes the sectioned correlation (set by choose_split), its hop length
    int corr_route = 0;  // 0: chosen by the plan, 1: direct lag sums (corr.cu), 2: sectioned FFT64 correlation (corr_os.cu)
    int cpr = 0;         // constant photometric ratio: centre coefficients of the terms t >= 1 not free
    bool pow2 = true;    // H and W are powers of two (mask wraps, radix-2 row transforms, every route available)
    int bsM = 0;         // W not a power of two: length of the M-point transforms of the chirp-z (Bluestein) row DFT
    int Lx = 0, Ly = 0;  // kernel extent along x / y (rectangular kernels); L = max(Lx, Ly) is the enclosing square
    bool reduced = false;   // the solved system is a reduction of the full square layout (cpr and / or Lx != Ly)
    int rshare = -1;     // solved index of the shared centre unknown under cpr
    int ns = 0;          // solved unknowns: n, or n - (FK - 1) under cpr
    int nimg = 0;        // spectrum stack depth per batch entry: nKa weighted-y images + S
    int nseq = 0;        // FK + 1 column sequences (kernel terms, then S)
    int E = 0;           // G entries per spectrum column: nseq*nseq*L
    int Sx = 1;          // x-range splits of the correlation kernel (partial sums added by lagsum)
    int nlb = 0;         // 8-lag blocks: ceil((L-1)/8)
    int lagchunk = sfft::kLagChunk;   // spectrum columns per partial sum (8, 16 or 32: enough CTAs to fill the machine)
    int nch = 0;         // column chunks of the lagsum partials
    int NC = 0;          // nKa*nBa*L columns of the moment GEMMs
    int ksplit = 1;      // K (x-range) splits of the second moment GEMM
    int nMom = 0;        // POLY: row power moments mu_a(x) = sum_y R(x,y) u_y^a kept per row
    int ksq = 1;         // K (y-range) splits of the first moment GEMM; its partial Q's are summed by the second
    int npairs = 0;      // FK(FK+1)/2
    int ldl = 0;         // leading dimension of the Cholesky factor buffer (>= n+1)
    int LT = 0;          // K extent per source row of the subtract contraction (nKa*L padded to 4)
    std::vector<int> kti, ktj, bti, btj;
    std::vector<sfft::Seq> seqs;
    std::vector<sfft::CorrJob> jobs;
    std::vector<sfft::LagUnit> units;
    sfft::DeviceTables dt;
    // lag-table layout (doubles per batch entry)
    size_t off_om = 0, off_th = 0, off_la = 0, off_de = 0, tab_size = 0;
    // workspace partition (device pointers into the caller's buffer)
    void *ws = nullptr; size_t ws_bytes = 0;
    double2 *rhat = nullptr; double2 *G = nullptr; double *lagpart = nullptr; double *tab = nullptr;
    double *Q = nullptr, *QS = nullptr, *LamC = nullptr, *mu = nullptr;
    double *M = nullptr, *rhs = nullptr, *Lf = nullptr, *Winv = nullptr, *dscale = nullptr, *kfold = nullptr, *ctab = nullptr;
    double2 *khat = nullptr;                    // [b][L*FK][Nh] row spectra of the pixel kernels (Fourier-route subtract)
    bool rhat_from_build = false;               // rhat[0..nKa) holds the spectra of the R given to the last build
    int reuse_spectra = 0;                      // caller's promise (sfft_plan_set_reuse_spectra): subtract R == build R
    bool host_call = false;                     // inside sfft_run_host*: build and subtract see the same staged pair
    int device = 0;                             // CUDA device the plan was created on
    double *coefr = nullptr;                    // [b][ns] reduced solution (cpr) before expansion to the full layout
    double *ybuf = nullptr;                     // [b][nblk*64] published blocks of the back substitution (solve.cu)
    // host-call staging: two slots so that the copies of one pair overlap the compute of another (sfft_run_host_async)
    double *stageR[2] = {nullptr, nullptr}, *stageS[2] = {nullptr, nullptr}, *stageD[2] = {nullptr, nullptr},
           *stageC[2] = {nullptr, nullptr};
    float *stageR32[2] = {nullptr, nullptr}, *stageS32[2] = {nullptr, nullptr}, *stageD32[2] = {nullptr, nullptr};
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;           // plan-owned copy streams
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
    int host_slot = 0;                                       // next staging slot (round robin)
    void *staging = nullptr; size_t staging_bytes = 0;       // caller-owned staging buffer (sfft_plan_set_host_staging)
    int *flag = nullptr;
    cudaStream_t stream = nullptr;
    cudaStream_t side = nullptr;                // plan-owned stream: the moment stage (HBM bound) runs beside the
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;   // tensor-bound lag correlation (fork/join on `stream`)
    bool built = false, solved = false;
    long launches = 0;
    int prof_steps = 0, prof_cur = -1;          // stage profiling (sfft_plan_profile)
    std::vector<cudaEvent_t> prof_events;       // [prof_steps][kProfMarks]
    std::string cuda_err;
    std::vector<double> decorr_host;            // sfft_decorrelate's copy of the caller's host tables (source of its uploads)
};

namespace sfft {
// stage launchers (each returns cudaError_t of the launch); all enqueue on p->stream
cudaError_t launch_rowfft_forward(sfft_plan *p, const double *dR, const double *dS);   // dS == nullptr: R rows only
cudaError_t launch_corr(sfft_plan *p);
bool corr_use_os(const sfft_plan *p);        // sectioned (overlap-save FFT64) lag correlation instead of direct lag sums
int corr_os_split(const sfft_plan *p);       // its x-range parts
int corr_os_hop(const sfft_plan *p);
cudaError_t launch_corr_os(sfft_plan *p);
cudaError_t launch_lagsum(sfft_plan *p);
cudaError_t launch_moments(sfft_plan *p, const double *dR, const double *dS);
cudaError_t launch_gather(sfft_plan *p);
cudaError_t launch_decorrelate(sfft_plan *p, const double *d_coef, const double *dD, double *dOut, int T, int nS,
                               const double *h_varS, int LG, const double *h_G, int nR, const double *h_varR, int LH,
                               const double *h_H);
cudaError_t launch_widen(sfft_plan *p, const float *src, double *dst, size_t count);     // float -> double (exact)
cudaError_t launch_narrow(sfft_plan *p, const double *src, float *dst, size_t count);    // double -> float (round to nearest)
cudaError_t launch_mask_fill(sfft_plan *p, const double *dR, const double *dS, double satR, double satS, int rd, int rb,
                             double *dRm, double *dSm, unsigned char *dmask);
cudaError_t launch_expand_coef(sfft_plan *p, const double *d_cr, double *d_coef);   // c = C c' (cpr)
cudaError_t launch_solve(sfft_plan *p, double *d_coef);
int solve_num_blocks(int n);     // 64-column panels of the Cholesky factorisation
int subtract_kpad(int nKa, int L);
void prof_mark(sfft_plan *p, int mark);
cudaError_t launch_subtract(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD);
cudaError_t launch_fold_coef(sfft_plan *p, const double *d_coef);          // delta-basis coefficients -> pixel kernels
bool subtract_use_fourier(const sfft_plan *p);                              // route choice of sfft_subtract
cudaError_t launch_subtract_fourier(sfft_plan *p, const double *d_coef, const double *dR, const double *dS, double *dD);

// C[M x N] (ldc) = alpha * A[M x K] (lda, row-major) * B + beta * C  on the FP64 tensor cores.
// bT = true : B given as [N x K] row-major (ldb)  ("A B^T");  false : B is [K x N] row-major.
// grid.z = nz problems with element strides sA, sB, sC; K may be split in `ksplit` parts, part q
// writing C + q*sCk (beta must then be 0).  lower = true : only tiles touching j <= i are computed.
struct GemmArgs {
    const double *A; const double *B; double *C;
    int M, N, K, lda, ldb, ldc;
    long long sA, sB, sC, sCk;
    int nz, ksplit;
    int kmodA;      // > 0: A's column index is k mod kmodA (B's K axis is kmodA-periodic stacks of partial operands)
    double alpha, beta;
    bool bT, lower;
};
cudaError_t launch_dgemm(sfft_plan *p, const GemmArgs &g);
}  // namespace sfft
