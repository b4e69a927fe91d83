// Plan construction, constant tables, workspace partition and the C ABI of libsfft_b200.
// The numerical stages live in rowfft.cu / corr.cu / gather.cu / solve.cu / subtract.cu.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "sfft_internal.h"

using namespace sfft;

namespace sfft {
// record profiling mark `m` of the current step on the plan's stream (no-op unless profiling)
void prof_mark(sfft_plan *p, int m) {
    if (p->prof_steps <= 0 || p->prof_cur < 0 || p->prof_cur >= p->prof_steps) return;
    cudaEventRecord(p->prof_events[(size_t)p->prof_cur * kProfMarks + m], p->stream);
}
}  // namespace sfft

namespace {

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }
size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }

int num_axis(int basis, int D) { return basis == SFFT_BASIS_POLY ? D + 1 : D + 4; }

// 1-D basis table tab[f][x] in long double precision, rounded once to double.
// POLY (Eqs. 2, 6 with the normalised coordinates of DESIGN g8): u^f, u = (2x+1)/N - 1.
// BSPLINE (Eqs. 8-9, DESIGN g13): cubic, clamped, D uniform interior knots, v = (x+0.5)/N,
// evaluated with the local-support triangular scheme (the 4 non-zero functions of the span).
std::vector<double> axis_table(int basis, int N, int D) {
    int nf = num_axis(basis, D);
    std::vector<double> tab((size_t)nf * N, 0.0);
    if (basis == SFFT_BASIS_POLY) {
        for (int x = 0; x < N; ++x) {
            long double u = (2.0L * x + 1.0L) / (long double)N - 1.0L, p = 1.0L;
            for (int f = 0; f < nf; ++f) { tab[(size_t)f * N + x] = (double)p; p *= u; }
        }
        return tab;
    }
    const int deg = 3, nspan = D + 1;
    std::vector<long double> U(nf + deg + 1);
    for (int q = 0; q <= deg; ++q) { U[q] = 0.0L; U[nf + deg - q] = 1.0L; }
    for (int q = 1; q <= D; ++q) U[deg + q] = (long double)q / (long double)nspan;
    for (int x = 0; x < N; ++x) {
        long double v = (x + 0.5L) / (long double)N;
        int span = deg;                                  // knot span index: U[span] <= v < U[span+1]
        while (span < nf - 1 && v >= U[span + 1]) ++span;
        long double Nb[deg + 1], left[deg + 1], right[deg + 1];
        Nb[0] = 1.0L;
        for (int j = 1; j <= deg; ++j) {
            left[j] = v - U[span + 1 - j];
            right[j] = U[span + j] - v;
            long double saved = 0.0L;
            for (int r = 0; r < j; ++r) {
                long double tmp = Nb[r] / (right[r + 1] + left[j - r]);
                Nb[r] = saved + right[r + 1] * tmp;
                saved = left[j - r] * tmp;
            }
            Nb[j] = saved;
        }
        for (int j = 0; j <= deg; ++j) tab[(size_t)(span - deg + j) * N + x] = (double)Nb[j];
    }
    return tab;
}

void term_list(int basis, int D, std::vector<int> &ti, std::vector<int> &tj) {
    ti.clear(); tj.clear();
    if (basis == SFFT_BASIS_POLY) {
        for (int i = 0; i <= D; ++i)
            for (int j = 0; j + i <= D; ++j) { ti.push_back(i); tj.push_back(j); }
    } else {
        for (int i = 0; i < D + 4; ++i)
            for (int j = 0; j < D + 4; ++j) { ti.push_back(i); tj.push_back(j); }
    }
}

template <typename T>
cudaError_t upload(T **dst, const T *src, size_t count) {
    cudaError_t e = cudaMalloc((void **)dst, std::max<size_t>(count, 1) * sizeof(T));
    if (e != cudaSuccess) return e;
    if (count) e = cudaMemcpy(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice);
    return e;
}

int pair_index(int FK, int t1, int t2) { return t1 * FK - t1 * (t1 - 1) / 2 + (t2 - t1); }  // t1 <= t2

// x-range splits of the correlation kernel: fill the 2 x 148 CTA slots evenly (partials are added in lagsum)
void choose_split(sfft_plan *p) {
    p->Sx = 1;
    const double slots = 2.0 * 148.0;
    double best = 1e300;
    for (int sx = 1; sx <= 8; sx *= 2) {
        if (p->H / sx < 32) break;
        double T = (double)(p->Nh / kCorrCols) * p->jobs.size() * p->nbatch * sx;
        double cost = ceil(T / slots) / sx * (1.0 + 0.02 * sx);     // mild penalty: G traffic grows with sx
        if (cost < best) { best = cost; p->Sx = sx; }
    }
    p->corr_os = corr_use_os(p);
    if (p->corr_os) { p->Sx = corr_os_split(p); p->os_hop = corr_os_hop(p); }
    // column chunks of the y-direction partial sums (lagsum.cu): enough CTAs to fill the machine
    p->lagchunk = kLagChunk;
    while (p->lagchunk > 8 && (long)((p->E + 127) / 128) * ((p->Nh + p->lagchunk) / p->lagchunk) * p->nbatch < 2 * 148)
        p->lagchunk /= 2;
    p->nch = (p->Nh + 1 + p->lagchunk - 1) / p->lagchunk;
    // y-range splits of the first moment GEMM (moments.cu): enough CTAs to fill the machine
    const long tiles = (long)((p->H + 63) / 64) * ((p->NC + 63) / 64) * p->nbatch;
    p->ksq = 1;
    while (p->basis != SFFT_BASIS_POLY && p->ksq < 8 && tiles * p->ksq < 4 * 148 && p->W / (2 * p->ksq) >= 256) p->ksq *= 2;
}

// Lags of G_{p,q} the normal system reads: L-1 between kernel terms (Omega, B5/B6), w against S (Theta, B13/B14),
// none for S with S.
int need_lag(const sfft_plan *p, int sp, int sq) {
    const bool ps = sp == p->FK, qs = sq == p->FK;
    return (ps && qs) ? -1 : ((ps || qs) ? p->w : p->L - 1);
}

void build_jobs(sfft_plan *p, const std::vector<double> &fK) {
    const int FK = p->FK, FB = p->FB, L = p->L, w = p->w, nO = 2 * L - 1, H = p->H;
    p->seqs.clear(); p->jobs.clear(); p->units.clear();
    // column sequences: kernel terms z_t = f_i(x) r_j(x,m), then S
    for (int t = 0; t < FK; ++t) p->seqs.push_back({p->ktj[t], p->kti[t]});
    const int seqS = FK;
    p->seqs.push_back({p->nKa, -1});
    p->nseq = FK + 1;
    p->E = p->nseq * p->nseq * L;
    // lag blocks: a shared lag-0 block plus blocks from lag 1 when L-1 is a multiple of 8, else blocks from lag 0
    const bool lag0blk = ((L - 1) % 8 == 0);
    p->nlb = lag0blk ? (L - 1) / 8 : (L + 7) / 8;
    p->npairs = FK * (FK + 1) / 2;
    p->off_om = 0;
    p->off_th = p->off_om + (size_t)p->npairs * nO * nO;
    p->off_la = p->off_th + (size_t)FK * L * L;
    p->off_de = p->off_la + (size_t)FK * FB * L * L;
    p->tab_size = p->off_de + FB;
    // x-support [lo, hi) of every sequence (B-spline x-factors are compactly supported; everything else is dense)
    std::vector<int> slo(p->nseq, 0), shi(p->nseq, H);
    if (p->basis == SFFT_BASIS_BSPLINE)
        for (int t = 0; t < FK; ++t) {
            const double *f = &fK[(size_t)p->kti[t] * H];
            int lo = 0, hi = H;
            while (lo < H && f[lo] == 0.0) ++lo;
            while (hi > lo && f[hi - 1] == 0.0) --hi;
            slo[t] = lo; shi[t] = hi;
        }
    // correlation jobs: (group of 8 M-side sequences) x (tile of knt N-side sequences, at most 16 blocks)
    const int knt = p->nlb == 0 ? 8 : std::min(8, (2 * kCorrBlk - (lag0blk ? 1 : 0)) / p->nlb);
    for (int m0 = 0; m0 < p->nseq; m0 += 8)
        for (int n0 = 0; n0 < p->nseq; n0 += knt) {
            CorrJob j{};
            const int mcnt = std::min(8, p->nseq - m0), ncnt = std::min(knt, p->nseq - n0);
            for (int q = 0; q < 8; ++q) { j.zslot[q] = kCorrZero; j.zseq[q] = -1; }
            // N side: planes 0..ncnt-1, blocks dealt to the two warp halves in turn
            struct Blk { int slot, seq, lag, nlag; };
            std::vector<Blk> blks;
            bool any0 = false;
            int Alo = H, Ahi = 0, Nlo = H, Nhi = 0, maxlag = 0;
            for (int q = 0; q < ncnt; ++q) {
                const int sq = n0 + q;
                int ml = -1;
                for (int r = 0; r < mcnt; ++r) ml = std::max(ml, need_lag(p, m0 + r, sq));
                if (ml < 0) continue;
                j.stage_slot[j.nstage] = q; j.stage_seq[j.nstage] = sq; ++j.nstage;
                Nlo = std::min(Nlo, slo[sq]); Nhi = std::max(Nhi, shi[sq]); maxlag = std::max(maxlag, ml);
                if (lag0blk) { j.zslot[q] = q; j.zseq[q] = sq; any0 = true; }
                for (int l0 = lag0blk ? 1 : 0; l0 <= ml; l0 += 8) blks.push_back({q, sq, l0, std::min(8, ml - l0 + 1)});
            }
            if (any0) blks.push_back({-1, -1, 0, 8});
            if (blks.empty()) continue;
            for (size_t i = 0; i < blks.size(); ++i) {
                const int h = (int)(i & 1), k = j.nblk[h]++;
                j.blk_slot[h][k] = blks[i].slot; j.blk_seq[h][k] = blks[i].seq;
                j.blk_lag[h][k] = blks[i].lag; j.blk_nlag[h][k] = blks[i].nlag;
            }
            for (int h = 0; h < 2; ++h)
                for (int k = j.nblk[h]; k < kCorrBlk; ++k) { j.blk_slot[h][k] = kCorrZero; j.blk_seq[h][k] = -1; j.blk_lag[h][k] = 0; j.blk_nlag[h][k] = 0; }
            // M side: share the plane of an N-side sequence, else an extra plane
            int extra = kCorrZero + 1;
            for (int h = 0; h < 2; ++h)
                for (int r = 0; r < 4; ++r) {
                    const int sq = m0 + 4 * h + r;
                    if (sq >= p->nseq) { j.mseq[h][r] = -1; j.mslot[h][r] = kCorrZero; continue; }
                    j.mseq[h][r] = sq;
                    Alo = std::min(Alo, slo[sq]); Ahi = std::max(Ahi, shi[sq]);
                    int slot = -1;
                    for (int k = 0; k < j.nstage; ++k) if (j.stage_seq[k] == sq) slot = j.stage_slot[k];
                    if (slot < 0) { slot = extra++; j.stage_slot[j.nstage] = slot; j.stage_seq[j.nstage] = sq; ++j.nstage; }
                    j.mslot[h][r] = slot;
                }
            // x-ranges where z_p(x) z_q(x + rho) can be non-zero: x in A with x + rho in N, directly or wrapped
            auto round4 = [&](int &lo, int &hi) { lo = std::max(0, lo & ~3); hi = std::min(H, (hi + 3) & ~3); };
            int lo1 = std::max(Alo, Nlo - maxlag), hi1 = std::min(Ahi, Nhi);
            int lo2 = std::max(Alo, H + Nlo - maxlag), hi2 = std::min(Ahi, H);      // x + rho - H in [Nlo, Nhi)
            round4(lo1, hi1); round4(lo2, hi2);
            const bool e1 = hi1 <= lo1, e2 = hi2 <= lo2;
            if (e1 && e2) { j.nrange = 1; j.xbeg[0] = 0; j.xend[0] = 4; }              // nothing overlaps: one all-zero step
            else if (e2 || (!e1 && lo2 <= hi1)) { j.nrange = 1; j.xbeg[0] = lo1; j.xend[0] = e2 ? hi1 : std::max(hi1, hi2); }
            else if (e1) { j.nrange = 1; j.xbeg[0] = lo2; j.xend[0] = hi2; }
            else { j.nrange = 2; j.xbeg[0] = lo1; j.xend[0] = hi1; j.xbeg[1] = lo2; j.xend[1] = hi2; }
            p->jobs.push_back(j);
        }
    // lag-table rows.  Negative x-lags use G_{p,q}(-rho) = conj G_{q,p}(rho): entry (q,p,|rho|) with eps negated.
    auto entry = [&](int pp, int qq, int rho) { return (pp * p->nseq + qq) * L + rho; };
    for (int tb = 0; tb < FK; ++tb)
        for (int t = tb; t < FK; ++t)
            for (int r = 0; r < nO; ++r) {
                int rho = r - (L - 1);
                int dst = (int)(p->off_om + ((size_t)pair_index(FK, tb, t) * nO + r) * nO);
                if (rho >= 0) p->units.push_back({entry(tb, t, rho), +1, L - 1, dst});
                else p->units.push_back({entry(t, tb, -rho), -1, L - 1, dst});
            }
    for (int tb = 0; tb < FK; ++tb)
        for (int r = 0; r < L; ++r) {
            int rho = r - w;
            int dst = (int)(p->off_th + ((size_t)tb * L + r) * L);
            if (rho >= 0) p->units.push_back({entry(tb, seqS, rho), +1, w, dst});
            else p->units.push_back({entry(seqS, tb, -rho), -1, w, dst});
        }
    p->NC = p->nKa * p->nBa * L;
    choose_split(p);
    p->ksplit = std::max(1, std::min(32, p->H / 64));
}

int fail_cuda(sfft_plan *p, cudaError_t e) {
    if (p) p->cuda_err = cudaGetErrorString(e);
    return SFFT_ERR_CUDA;
}

void free_tables(sfft_plan *p) {
    DeviceTables &d = p->dt;
    cudaFree(d.xwt); cudaFree(d.gK); cudaFree(d.gB); cudaFree(d.twW); cudaFree(d.twM); cudaFree(d.chirp); cudaFree(d.bhat); cudaFree(d.lagtw); cudaFree(d.cy); cudaFree(d.fx); cudaFree(d.cq); cudaFree(d.cwr);
    cudaFree(d.phi0);
    cudaFree(d.seqs); cudaFree(d.jobs); cudaFree(d.units);
    cudaFree(d.ridx); cudaFree(d.fmap);
    cudaFree(d.kdec); cudaFree(d.kti); cudaFree(d.ktj); cudaFree(d.bti); cudaFree(d.btj);
    d = DeviceTables();
}

struct WsLayout {
    size_t rhat, G, lagpart, tab, Q, QS, LamC, mu, M, rhs, Lf, Winv, dscale, coefr, ybuf, kfold, ctab, khat, flag, total;
};
struct StagingLayout { size_t stR[2], stS[2], stD[2], stC[2], stR32[2], stS32[2], stD32[2], total; };

WsLayout ws_layout(const sfft_plan *p) {
    WsLayout l{};
    size_t nb = p->nbatch, n = p->n, off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    l.rhat = take(nb * p->nimg * (size_t)p->H * p->Nh * sizeof(double2));
    l.G = take(nb * p->Sx * (size_t)(p->Nh + 1) * p->E * sizeof(double2));
    l.lagpart = take(nb * p->nch * (size_t)p->L * 2 * p->E * sizeof(double));
    l.tab = take(nb * p->tab_size * sizeof(double));
    l.Q = take(nb * p->ksq * (size_t)p->H * p->NC * sizeof(double));
    l.QS = take(nb * (size_t)p->H * p->nBa * sizeof(double));
    l.LamC = take(nb * p->ksq * p->ksplit * (size_t)p->NC * p->NC * sizeof(double));
    l.mu = take(nb * (size_t)p->H * p->nMom * sizeof(double));
    l.M = take(nb * n * n * sizeof(double));
    l.rhs = take(nb * n * sizeof(double));
    l.Lf = take(nb * (n + 1) * (size_t)p->ldl * sizeof(double));
    l.Winv = take(nb * (size_t)solve_num_blocks(p->n) * 64 * 64 * sizeof(double));
    l.dscale = take(nb * n * sizeof(double));
    l.coefr = take(nb * n * sizeof(double));
    l.ybuf = take(nb * (size_t)solve_num_blocks(p->n) * 64 * sizeof(double));
    l.kfold = take(nb * (size_t)p->FK * p->L * p->L * sizeof(double));
    // only the subtract route the plan takes gets its table
    l.ctab = take(subtract_use_fourier(p) ? 0 : nb * (size_t)p->H * p->L * p->LT * sizeof(double));
    l.khat = take(subtract_use_fourier(p) ? nb * (size_t)p->L * p->FK * p->Nh * sizeof(double2) : 0);
    l.flag = take((nb + 1) * sizeof(int) * 2);      // per system (first bad pivot, spare), then the back substitution's ticket
    l.total = off;
    return l;
}

// staging area of the host-buffer entry points: two slots of (R, S, D, coefficients)
StagingLayout staging_layout(const sfft_plan *p) {
    StagingLayout l{};
    size_t nb = p->nbatch, P = (size_t)p->H * p->W, off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    for (int q = 0; q < 2; ++q) {
        l.stR[q] = take(nb * P * sizeof(double));
        l.stS[q] = take(nb * P * sizeof(double));
        l.stD[q] = take(nb * P * sizeof(double));
        l.stC[q] = take(nb * (size_t)p->n * sizeof(double));
        l.stR32[q] = take(nb * P * sizeof(float));          // FP32-storage entry points
        l.stS32[q] = take(nb * P * sizeof(float));
        l.stD32[q] = take(nb * P * sizeof(float));
    }
    l.total = off;
    return l;
}

// Solved unknowns of a reduced system, in the order of the full (square) layout:
//   rectangular kernel: the entries with |alpha| > (Lx-1)/2 or |beta| > (Ly-1)/2 are fixed at zero;
//   constant photometric ratio (DESIGN g20): the centre entries of the terms t >= 1 are not free
//   (POLY: zero; BSPLINE: equal to the centre entry of t = 0, the shared unknown at solved index `rshare`).
// ridx[r] = full index of solved unknown r;  fmap[k] = solved index of full unknown k, or -1 (zero).
cudaError_t build_reduction(sfft_plan *p) {
    const int L = p->L, w = p->w, LL = L * L, wx = (p->Lx - 1) / 2, wy = (p->Ly - 1) / 2, a0 = w * L + w;
    std::vector<int> ridx, fmap(p->n, -1);
    p->rshare = -1;
    for (int k = 0; k < p->n; ++k) {
        if (k < p->FK * LL) {
            const int t = k / LL, a = k % LL, al = a / L - w, be = a % L - w;
            if (al < -wx || al > wx || be < -wy || be > wy) continue;
            if (p->cpr && a == a0 && t > 0) continue;
            if (p->cpr && a == a0) p->rshare = (int)ridx.size();
        }
        fmap[k] = (int)ridx.size();
        ridx.push_back(k);
    }
    if (p->cpr && p->basis != SFFT_BASIS_POLY)
        for (int t = 1; t < p->FK; ++t) fmap[t * LL + a0] = p->rshare;
    p->ns = (int)ridx.size();
    p->reduced = p->ns != p->n;
    cudaFree(p->dt.ridx); cudaFree(p->dt.fmap);
    p->dt.ridx = p->dt.fmap = nullptr;
    cudaError_t e = upload(&p->dt.ridx, ridx.data(), ridx.size());
    if (e == cudaSuccess) e = upload(&p->dt.fmap, fmap.data(), fmap.size());
    return e;
}

// a plan is tied to the device it was created on
bool wrong_device(const sfft_plan *p) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return true; }
    return dev != p->device;
}

}  // namespace

extern "C" {

int sfft_plan_create(sfft_plan **out, int H, int W, int L, int DK, int DB, int basis) {
    return sfft_plan_create_rect(out, H, W, L, L, DK, DB, basis);
}

int sfft_plan_create_rect(sfft_plan **out, int H, int W, int L0, int L1, int DK, int DB, int basis) {
    if (!out) return SFFT_ERR_INVALID_ARG;
    *out = nullptr;
    if (H < 32 || H > 8192 || W < 64 || W > 8192 || (W & 1)) return SFFT_ERR_INVALID_ARG;
    const bool pow2 = is_pow2(H) && is_pow2(W);
    if (!is_pow2(W) && W > 4096) return SFFT_ERR_INVALID_ARG;      // chirp-z row transform: M = 2^k >= W - 1, M <= 4096
    if (L0 < 1 || L0 > 33 || (L0 % 2) == 0 || L1 < 1 || L1 > 33 || (L1 % 2) == 0) return SFFT_ERR_INVALID_ARG;
    const int L = std::max(L0, L1);      // every table is built for the enclosing square; the gather keeps the rectangle
    if (2 * L - 1 > std::min(H, W)) return SFFT_ERR_INVALID_ARG;
    if (DK < 0 || DB < 0 || DK > 8 || DB > 8) return SFFT_ERR_INVALID_ARG;
    if (basis != SFFT_BASIS_POLY && basis != SFFT_BASIS_BSPLINE) return SFFT_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return SFFT_ERR_CUDA; }

    sfft_plan *p = new (std::nothrow) sfft_plan();
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (cudaGetDevice(&p->device) != cudaSuccess) { cudaGetLastError(); delete p; return SFFT_ERR_CUDA; }
    p->H = H; p->W = W; p->L = L; p->w = (L - 1) / 2; p->DK = DK; p->DB = DB; p->basis = basis;
    p->Lx = L0; p->Ly = L1;
    p->pow2 = pow2;
    if (!is_pow2(W)) { p->bsM = 512; while (p->bsM < W - 1) p->bsM *= 2; }
    p->Nh = W / 2;
    p->nKa = num_axis(basis, DK); p->nBa = num_axis(basis, DB);
    term_list(basis, DK, p->kti, p->ktj);
    term_list(basis, DB, p->bti, p->btj);
    p->FK = (int)p->kti.size(); p->FB = (int)p->bti.size();
    p->n = p->FK * L * L + p->FB;
    p->ns = p->n;
    // frames that are not powers of two need the sectioned lag correlation (polynomial basis, at most 8 column
    // sequences, DK <= 2); their subtract takes either route (chirp-z inverse rows on the Fourier route)
    if (!pow2 && (basis != SFFT_BASIS_POLY || p->FK + 1 > 8 || p->nKa > 3)) { delete p; return SFFT_ERR_INVALID_ARG; }
    p->nimg = p->nKa + 1;
    p->ldl = (p->n + 1 + 7) & ~7;
    p->LT = subtract_kpad(p->nKa, L);
    p->nMom = basis == SFFT_BASIS_POLY ? DK + DB + 1 : 0;

    // ---- constant tables (host, long double where it matters) ----
    std::vector<double> fK = axis_table(basis, H, DK), gK = axis_table(basis, W, DK);
    std::vector<double> fB = axis_table(basis, H, DB), gB = axis_table(basis, W, DB);
    build_jobs(p, fK);
    std::vector<double> xwt((size_t)(p->nKa + p->nBa) * H);
    std::copy(fK.begin(), fK.end(), xwt.begin());
    std::copy(fB.begin(), fB.end(), xwt.begin() + (size_t)p->nKa * H);
    std::vector<long double> cw(W), sw(W);
    std::vector<double2> twW(W);
    const long double twopi = 6.283185307179586476925286766559L;
    for (int k = 0; k < W; ++k) {
        // exact octant symmetry is not needed; cosl/sinl are accurate to long-double ulp
        cw[k] = cosl(twopi * k / W); sw[k] = -sinl(twopi * k / W);
        twW[k] = make_double2((double)cw[k], (double)sw[k]);
    }
    // y-direction pruned inverse DFT weights (lagsum.cu): (w_m cos, w_m sin)(2 pi m k / W) / W
    std::vector<double2> lagtw((size_t)(p->Nh + 1) * L);
    for (int m = 0; m <= p->Nh; ++m)
        for (int k = 0; k < L; ++k) {
            int idx = (int)(((long long)m * k) % W);
            long double wm = (m == 0 || m == p->Nh) ? 1.0L : 2.0L;
            lagtw[(size_t)m * L + k] = make_double2((double)(wm * cw[idx] / W), (double)(wm * -sw[idx] / W));
        }
    // moment-GEMM operands (moments.cu): products of a kernel and a shifted background basis function
    const int wl = p->w;
    // (cy is the operand of the first moment contraction, used by the B-spline path only: the polynomial path
    // replaces that contraction by row power moments, tables cq / cwr below)
    std::vector<double> cy(basis == SFFT_BASIS_POLY ? 0 : (size_t)p->NC * W), fx((size_t)p->NC * H);
    for (int jb = 0; jb < p->nKa && basis != SFFT_BASIS_POLY; ++jb)
        for (int j = 0; j < p->nBa; ++j)
            for (int b = 0; b < L; ++b) {
                double *row = &cy[((size_t)(jb * p->nBa + j) * L + b) * W];
                for (int y = 0; y < W; ++y) row[y] = gK[(size_t)jb * W + y] * gB[(size_t)j * W + ((y + b - wl + W) % W)];
            }
    for (int ib = 0; ib < p->nKa; ++ib)
        for (int i = 0; i < p->nBa; ++i)
            for (int a = 0; a < L; ++a) {
                double *row = &fx[((size_t)(ib * p->nBa + i) * L + a) * H];
                for (int x = 0; x < H; ++x) row[x] = fK[(size_t)ib * H + x] * fB[(size_t)i * H + ((x + a - wl + H) % H)];
            }
    // POLY shortcut of the first moment contraction (moments.cu): u(y+beta) = u(y) + beta*delta away from the wrap, so
    //   Q[x][(jb,j,beta)] = sum_k C(j,k) (beta delta)^(j-k) mu_{jb+k}(x) + sum_{wrapping y} R(x,y) u^jb [u(y')^j - (u + beta delta)^j]
    std::vector<double> cq, cwr;
    if (basis == SFFT_BASIS_POLY) {
        const int A = p->nMom;
        cq.assign((size_t)p->NC * A, 0.0); cwr.assign((size_t)p->NC * std::max(wl, 1), 0.0);
        auto uy = [&](int y) { return (2.0L * y + 1.0L) / (long double)W - 1.0L; };
        const long double delta = 2.0L / (long double)W;
        for (int jb = 0; jb < p->nKa; ++jb)
            for (int j = 0; j < p->nBa; ++j)
                for (int b = 0; b < L; ++b) {
                    const int c = (jb * p->nBa + j) * L + b, beta = b - wl;
                    long double binom = 1.0L;                       // C(j,k)
                    for (int k = 0; k <= j; ++k) {
                        cq[(size_t)c * A + jb + k] = (double)(binom * powl(beta * delta, j - k));
                        binom = binom * (j - k) / (k + 1);
                    }
                    for (int q = 0; q < std::abs(beta); ++q) {
                        const int y = beta > 0 ? W - beta + q : q, yw = beta > 0 ? y + beta - W : y + beta + W;
                        cwr[(size_t)c * wl + q] = (double)(powl(uy(y), jb) * (powl(uy(yw), j) - powl(uy(y) + beta * delta, j)));
                    }
                }
    }
    // M_bb = sum_x f_ib f_i * sum_y g_jb g_j  (Eq. 22 / B11 at lag 0; separable, plan constant)
    std::vector<double> phi0((size_t)p->FB * p->FB);
    {
        std::vector<long double> sx((size_t)p->nBa * p->nBa), sy((size_t)p->nBa * p->nBa);
        for (int a = 0; a < p->nBa; ++a)
            for (int b = 0; b < p->nBa; ++b) {
                long double ax = 0.0L, ay = 0.0L;
                for (int x = 0; x < H; ++x) ax += (long double)fB[(size_t)a * H + x] * fB[(size_t)b * H + x];
                for (int y = 0; y < W; ++y) ay += (long double)gB[(size_t)a * W + y] * gB[(size_t)b * W + y];
                sx[a * p->nBa + b] = ax; sy[a * p->nBa + b] = ay;
            }
        for (int sb = 0; sb < p->FB; ++sb)
            for (int s = 0; s < p->FB; ++s)
                phi0[(size_t)sb * p->FB + s] =
                    (double)(sx[p->bti[sb] * p->nBa + p->bti[s]] * sy[p->btj[sb] * p->nBa + p->btj[s]]);
    }

    // chirp-z (Bluestein) row DFT for W not a power of two: with N = W/2 and c[n] = exp(-i pi n^2 / N),
    //   Z[k] = sum_n z[n] exp(-2 pi i n k / N) = c[k] sum_n (z[n] c[n]) conj(c[k-n]),
    // a circular convolution of length M >= 2N - 1 run with two M-point transforms (rowfft.cu)
    std::vector<double2> twM, chirp, bhat;
    if (p->bsM) {
        const int M = p->bsM, N = W / 2;
        const long double pi = 3.141592653589793238462643383279L;
        twM.resize(2 * (size_t)M); chirp.resize(N); bhat.resize(M);
        for (int k = 0; k < 2 * M; ++k) twM[k] = make_double2((double)cosl(pi * k / M), (double)-sinl(pi * k / M));
        std::vector<long double> br(M, 0.0L), bi(M, 0.0L), tc(M), ts(M);
        for (int n = 0; n < N; ++n) {
            const long long q = ((long long)n * n) % (2LL * N);          // n^2 mod 2N: the angle is exact
            const long double cr = cosl(pi * q / N), ci = sinl(pi * q / N);
            chirp[n] = make_double2((double)cr, (double)-ci);
            br[n] = cr; bi[n] = ci;
            if (n) { br[M - n] = cr; bi[M - n] = ci; }
        }
        for (int k = 0; k < M; ++k) { tc[k] = cosl(2.0L * pi * k / M); ts[k] = -sinl(2.0L * pi * k / M); }
        for (int q = 0; q < M; ++q) {
            long double sr = 0.0L, si = 0.0L;
            for (int m = 0; m < M; ++m) {
                if (br[m] == 0.0L && bi[m] == 0.0L) continue;
                const int idx = (int)(((long long)q * m) & (M - 1));
                sr += br[m] * tc[idx] - bi[m] * ts[idx];
                si += br[m] * ts[idx] + bi[m] * tc[idx];
            }
            bhat[q] = make_double2((double)sr, (double)si);
        }
    }

    cudaError_t e = cudaSuccess;
    DeviceTables &d = p->dt;
#define UP(dst, vec) if (e == cudaSuccess) e = upload(&d.dst, vec.data(), vec.size())
    UP(xwt, xwt); UP(gK, gK); UP(gB, gB); UP(twW, twW); UP(twM, twM); UP(chirp, chirp); UP(bhat, bhat); UP(lagtw, lagtw); UP(cy, cy); UP(fx, fx); UP(cq, cq); UP(cwr, cwr); UP(phi0, phi0);
    std::vector<int> kdec((size_t)p->FK * L * L);
    for (int t = 0; t < p->FK; ++t)
        for (int a = 0; a < L * L; ++a) kdec[(size_t)t * L * L + a] = (t << 16) | ((a / L) << 8) | (a % L);
    UP(kdec, kdec);
    if (e == cudaSuccess) e = build_reduction(p);
    UP(seqs, p->seqs); UP(jobs, p->jobs); UP(units, p->units);
    UP(kti, p->kti); UP(ktj, p->ktj); UP(bti, p->bti); UP(btj, p->btj);
#undef UP
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking);
    for (int q = 0; q < 2 && e == cudaSuccess; ++q) {
        e = cudaEventCreateWithFlags(&p->ev_in[q], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_done[q], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_out[q], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { sfft_plan_destroy(p); cudaGetLastError(); return SFFT_ERR_CUDA; }
    *out = p;
    return SFFT_OK;
}

int sfft_plan_set_batch(sfft_plan *p, int nbatch) {
    if (!p || nbatch < 1 || nbatch > 65535) return SFFT_ERR_INVALID_ARG;
    p->nbatch = nbatch; p->ws = nullptr; p->ws_bytes = 0; p->built = p->solved = false;
    p->staging = nullptr; p->staging_bytes = 0;
    choose_split(p);
    return SFFT_OK;
}

int sfft_plan_set_const_phot_ratio(sfft_plan *p, int on) {
    if (!p || (on != 0 && on != 1)) return SFFT_ERR_INVALID_ARG;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    p->cpr = on;
    p->built = p->solved = false;
    cudaError_t e = build_reduction(p);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return SFFT_OK;
}

int sfft_plan_num_solved(const sfft_plan *p) { return p ? p->ns : -1; }

int sfft_plan_set_corr_route(sfft_plan *p, int route) {
    if (!p || route < 0 || route > 2) return SFFT_ERR_INVALID_ARG;
    p->corr_route = route;
    if ((route == 2 && !corr_use_os(p)) || (route == 1 && !p->pow2)) { p->corr_route = 0; return SFFT_ERR_INVALID_ARG; }
    p->ws = nullptr; p->ws_bytes = 0; p->built = p->solved = false;      // the workspace partition depends on the split
    choose_split(p);
    return SFFT_OK;
}

int sfft_plan_set_stream(sfft_plan *p, void *stream) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    p->stream = (cudaStream_t)stream;
    return SFFT_OK;
}

int sfft_plan_num_unknowns(const sfft_plan *p) { return p ? p->n : -1; }
int sfft_plan_num_kernel_terms(const sfft_plan *p) { return p ? p->FK : -1; }
int sfft_plan_num_background_terms(const sfft_plan *p) { return p ? p->FB : -1; }

size_t sfft_plan_workspace_bytes(const sfft_plan *p) { return p ? ws_layout(p).total : 0; }

int sfft_plan_set_workspace(sfft_plan *p, void *d_ws, size_t bytes) {
    if (!p || !d_ws) return SFFT_ERR_INVALID_ARG;
    WsLayout l = ws_layout(p);
    if (bytes < l.total || ((uintptr_t)d_ws & 255)) return SFFT_ERR_WORKSPACE;
    char *b = (char *)d_ws;
    p->ws = d_ws; p->ws_bytes = bytes;
    p->rhat = (double2 *)(b + l.rhat); p->G = (double2 *)(b + l.G); p->lagpart = (double *)(b + l.lagpart); p->tab = (double *)(b + l.tab);
    p->Q = (double *)(b + l.Q); p->QS = (double *)(b + l.QS); p->LamC = (double *)(b + l.LamC); p->mu = (double *)(b + l.mu);
    p->M = (double *)(b + l.M); p->rhs = (double *)(b + l.rhs); p->Lf = (double *)(b + l.Lf); p->Winv = (double *)(b + l.Winv);
    p->dscale = (double *)(b + l.dscale); p->coefr = (double *)(b + l.coefr); p->ybuf = (double *)(b + l.ybuf); p->kfold = (double *)(b + l.kfold); p->ctab = (double *)(b + l.ctab); p->khat = (double2 *)(b + l.khat); p->flag = (int *)(b + l.flag);
    p->built = p->solved = false;
    p->rhat_from_build = false;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    // "no failure" marks: sfft_plan_status may be asked before the first build has cleared them
    if (cudaMemsetAsync(p->flag, 0xff, sizeof(int) * 2 * p->nbatch, p->stream) != cudaSuccess) return fail_cuda(p, cudaGetLastError());
    if (!p->corr_os) {
        // the direct lag-sum kernel never writes the (S, S) pair and the lags beyond w against S, which the
        // y-direction sums read along with everything else (their results are not used): keep those entries defined
        if (wrong_device(p)) return SFFT_ERR_STATE;
        cudaError_t e = cudaMemsetAsync(p->G, 0, l.lagpart - l.G, p->stream);
        if (e != cudaSuccess) return fail_cuda(p, e);
    }
    return SFFT_OK;
}

size_t sfft_plan_host_staging_bytes(const sfft_plan *p) { return p ? staging_layout(p).total : 0; }

int sfft_plan_set_host_staging(sfft_plan *p, void *d_buf, size_t bytes) {
    if (!p || !d_buf) return SFFT_ERR_INVALID_ARG;
    StagingLayout l = staging_layout(p);
    if (bytes < l.total || ((uintptr_t)d_buf & 255)) return SFFT_ERR_WORKSPACE;
    char *b = (char *)d_buf;
    p->staging = d_buf; p->staging_bytes = bytes;
    for (int q = 0; q < 2; ++q) {
        p->stageR[q] = (double *)(b + l.stR[q]); p->stageS[q] = (double *)(b + l.stS[q]);
        p->stageD[q] = (double *)(b + l.stD[q]); p->stageC[q] = (double *)(b + l.stC[q]);
        p->stageR32[q] = (float *)(b + l.stR32[q]); p->stageS32[q] = (float *)(b + l.stS32[q]);
        p->stageD32[q] = (float *)(b + l.stD32[q]);
    }
    p->host_slot = 0;
    return SFFT_OK;
}

int sfft_plan_set_reuse_spectra(sfft_plan *p, int on) {
    if (!p || (on != 0 && on != 1)) return SFFT_ERR_INVALID_ARG;
    p->reuse_spectra = on;
    return SFFT_OK;
}

int sfft_build_system(sfft_plan *p, const double *d_R, const double *d_S) {
    if (!p || !d_R || !d_S) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    p->built = p->solved = false;
    cudaError_t e = cudaMemsetAsync(p->flag, 0xff, sizeof(int) * 2 * p->nbatch, p->stream);  // -1 = no failure
    if (p->prof_steps > 0) p->prof_cur = p->prof_cur + 1;   // a build opens the next profiled step
    prof_mark(p, 0);
    // The moment stage depends only on (R, S): unless stages are being timed it is forked onto the plan's
    // side stream, where its streaming passes run beside the tensor-bound lag correlation, and joined
    // before the gather.
    const bool fork = p->side && p->prof_steps <= 0;
    if (fork && e == cudaSuccess) {
        e = cudaEventRecord(p->ev_fork, p->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->side, p->ev_fork, 0);
        if (e == cudaSuccess) {
            cudaStream_t main = p->stream;
            p->stream = p->side;
            e = launch_moments(p, d_R, d_S);
            p->stream = main;
        }
        if (e == cudaSuccess) e = cudaEventRecord(p->ev_join, p->side);
    }
    if (e == cudaSuccess) e = launch_rowfft_forward(p, d_R, d_S);
    p->rhat_from_build = (e == cudaSuccess);
    prof_mark(p, 1);
    if (e == cudaSuccess) e = launch_corr(p);
    prof_mark(p, 2);
    if (e == cudaSuccess) e = launch_lagsum(p);
    prof_mark(p, 3);
    if (!fork && e == cudaSuccess) e = launch_moments(p, d_R, d_S);
    if (fork && e == cudaSuccess) e = cudaStreamWaitEvent(p->stream, p->ev_join, 0);
    prof_mark(p, 4);
    if (e == cudaSuccess) e = launch_gather(p);
    prof_mark(p, 5);
    if (e != cudaSuccess) return fail_cuda(p, e);
    p->built = true;
    return SFFT_OK;
}

int sfft_plan_profile(sfft_plan *p, int nsteps) {
    if (!p || nsteps < 0 || nsteps > 4096) return SFFT_ERR_INVALID_ARG;
    for (cudaEvent_t ev : p->prof_events) cudaEventDestroy(ev);
    p->prof_events.clear();
    p->prof_steps = nsteps; p->prof_cur = -1;
    for (int i = 0; i < nsteps * kProfMarks; ++i) {
        cudaEvent_t ev;
        if (cudaEventCreate(&ev) != cudaSuccess) return fail_cuda(p, cudaGetLastError());
        p->prof_events.push_back(ev);
    }
    return SFFT_OK;
}

int sfft_plan_profile_read(sfft_plan *p, double *ms, int *nrecorded) {
    if (!p || !ms) return SFFT_ERR_INVALID_ARG;
    cudaError_t e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e);
    int nrec = std::min(p->prof_cur + 1, p->prof_steps);
    if (nrecorded) *nrecorded = nrec;
    // stages: 0 rowfft, 1 corr, 2 lagsum, 3 moments, 4 gather, 5 solve, 6 subtract-prep, 7 subtract, and the two halves
    // of 7 on the Fourier route (mark 11 lies between them; never recorded on the direct route): 8 FIR, 9 inverse rows
    static const int from[SFFT_NUM_STAGES] = {0, 1, 2, 3, 4, 6, 8, 9, 9, 11}, to[SFFT_NUM_STAGES] = {1, 2, 3, 4, 5, 7, 9, 10, 11, 10};
    for (int s = 0; s < nrec; ++s)
        for (int g = 0; g < SFFT_NUM_STAGES; ++g) {
            float t = 0.f;
            cudaError_t q = cudaEventElapsedTime(&t, p->prof_events[(size_t)s * kProfMarks + from[g]],
                                                 p->prof_events[(size_t)s * kProfMarks + to[g]]);
            ms[(size_t)s * SFFT_NUM_STAGES + g] = (q == cudaSuccess) ? (double)t : -1.0;
            if (q != cudaSuccess) cudaGetLastError();
        }
    return SFFT_OK;
}

int sfft_get_system(const sfft_plan *p, const double **d_M, const double **d_rhs, int *ld) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    if (!p->built) return SFFT_ERR_STATE;
    if (d_M) *d_M = p->M;
    if (d_rhs) *d_rhs = p->rhs;
    if (ld) *ld = p->ns;
    return SFFT_OK;
}

int sfft_get_lag_table(const sfft_plan *p, int which, const double **d_table, size_t *count, size_t *batch_stride) {
    if (!p || which < 0 || which > 3) return SFFT_ERR_INVALID_ARG;
    if (!p->built) return SFFT_ERR_STATE;
    size_t off[5] = {p->off_om, p->off_th, p->off_la, p->off_de, p->tab_size};
    if (d_table) *d_table = p->tab + off[which];
    if (count) *count = off[which + 1] - off[which];
    if (batch_stride) *batch_stride = p->tab_size;
    return SFFT_OK;
}

int sfft_solve(sfft_plan *p, double *d_coef) {
    if (!p || !d_coef) return SFFT_ERR_INVALID_ARG;
    if (!p->built || wrong_device(p)) return SFFT_ERR_STATE;
    prof_mark(p, 6);
    cudaError_t e = launch_solve(p, d_coef);
    prof_mark(p, 7);
    if (e != cudaSuccess) return fail_cuda(p, e);
    p->solved = true;
    return SFFT_OK;
}

int sfft_subtract(sfft_plan *p, const double *d_coef, const double *d_R, const double *d_S, double *d_D) {
    if (!p || !d_coef || !d_R || !d_S || !d_D) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    prof_mark(p, 8);
    cudaError_t e = launch_subtract(p, d_coef, d_R, d_S, d_D);
    prof_mark(p, 10);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return SFFT_OK;
}

int sfft_mask_fill(sfft_plan *p, const double *d_R, const double *d_S, double sat_R, double sat_S, int rd, int rb,
                   double *d_Rm, double *d_Sm, unsigned char *d_mask) {
    if (!p || !d_R || !d_S || !d_Rm || !d_Sm || !d_mask) return SFFT_ERR_INVALID_ARG;
    if (rd < 0 || rd > 64 || rb < 1 || rb > 128 || !(sat_R == sat_R) || !(sat_S == sat_S)) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    p->rhat_from_build = false;                 // the spectrum area is used as scratch
    cudaError_t e = launch_mask_fill(p, d_R, d_S, sat_R, sat_S, rd, rb, d_Rm, d_Sm, d_mask);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return SFFT_OK;
}

int sfft_decorrelate(sfft_plan *p, const double *d_coef, const double *d_D, double *d_Ddc, int tile, int nS,
                     const double *h_varS, int LG, const double *h_G, int nR, const double *h_varR, int LH,
                     const double *h_H) {
    if (!p || !d_coef || !d_D || !d_Ddc || !h_varS || !h_G || !h_varR || !h_H) return SFFT_ERR_INVALID_ARG;
    if (!is_pow2(tile) || tile < 32 || tile > 512 || p->H % tile || p->W % tile || p->L > tile) return SFFT_ERR_INVALID_ARG;
    if (nS < 1 || nR < 1 || nS > 64 || nR > 64 || LG < 1 || LH < 1 || !(LG & 1) || !(LH & 1) || LG > tile || LH > tile ||
        LG > 65 || LH > 65)
        return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    const size_t P = (size_t)p->H * p->W, area = (size_t)p->nbatch * p->nimg * P * sizeof(double);
    const size_t need = (size_t)p->nbatch * P * sizeof(double) + (size_t)tile * sizeof(double2) +
                        2 * (size_t)tile * (tile / 2 + 1) * sizeof(double) +
                        ((size_t)nS * LG * LG + nS + (size_t)nR * LH * LH + nR) * sizeof(double);
    if (need > area) return SFFT_ERR_WORKSPACE;
    p->rhat_from_build = false;                 // the spectrum area is used as scratch
    cudaError_t e = launch_decorrelate(p, d_coef, d_D, d_Ddc, tile, nS, h_varS, LG, h_G, nR, h_varR, LH, h_H);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return SFFT_OK;
}

int sfft_plan_status(sfft_plan *p, int *info) {
    if (info) *info = -1;
    if (!p) return SFFT_ERR_INVALID_ARG;
    cudaError_t e = cudaStreamSynchronize(p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e);
    if (!p->ws) return SFFT_OK;
    std::vector<int> h(2 * (size_t)p->nbatch);
    e = cudaMemcpy(h.data(), p->flag, h.size() * sizeof(int), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(p, e);
    for (int b = 0; b < p->nbatch; ++b)
        if (h[2 * b] >= 0) {
            if (info) *info = b * p->ns + h[2 * b];
            return SFFT_ERR_NOT_SPD;
        }
    return SFFT_OK;
}

// Common body of the host-buffer entry points; f32 = images stored as float on the host.
static int run_host_async_any(sfft_plan *p, const void *h_R, const void *h_S, void *h_D, double *h_coef, bool f32) {
    if (!p || !h_R || !h_S) return SFFT_ERR_INVALID_ARG;
    if (!p->ws || !p->staging) return SFFT_ERR_WORKSPACE;
    if (wrong_device(p)) return SFFT_ERR_STATE;
    const int q = p->host_slot;
    p->host_slot ^= 1;
    const size_t npix = (size_t)p->nbatch * p->H * p->W;
    const size_t img = npix * (f32 ? sizeof(float) : sizeof(double));
    // H2D on the copy stream, after the previous user of this slot (two calls ago) has finished computing
    cudaError_t e = cudaStreamWaitEvent(p->s_h2d, p->ev_done[q], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(f32 ? (void *)p->stageR32[q] : (void *)p->stageR[q], h_R, img, cudaMemcpyHostToDevice, p->s_h2d);
    if (e == cudaSuccess) e = cudaMemcpyAsync(f32 ? (void *)p->stageS32[q] : (void *)p->stageS[q], h_S, img, cudaMemcpyHostToDevice, p->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(p->ev_in[q], p->s_h2d);
    // compute on the plan's stream once the inputs are in and the slot's previous result has left
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->stream, p->ev_in[q], 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->stream, p->ev_out[q], 0);
    if (f32 && e == cudaSuccess) e = launch_widen(p, p->stageR32[q], p->stageR[q], npix);
    if (f32 && e == cudaSuccess) e = launch_widen(p, p->stageS32[q], p->stageS[q], npix);
    if (e != cudaSuccess) return fail_cuda(p, e);
    int st = sfft_build_system(p, p->stageR[q], p->stageS[q]);
    if (st == SFFT_OK) st = sfft_solve(p, p->stageC[q]);
    p->host_call = true;        // the subtract sees the very pair the build transformed: its spectra are reused
    if (st == SFFT_OK) st = sfft_subtract(p, p->stageC[q], p->stageR[q], p->stageS[q], p->stageD[q]);
    p->host_call = false;
    if (st != SFFT_OK) return st;
    e = (f32 && h_D) ? launch_narrow(p, p->stageD[q], p->stageD32[q], npix) : cudaSuccess;
    if (e == cudaSuccess) e = cudaEventRecord(p->ev_done[q], p->stream);
    // D2H on the other copy stream
    if (e == cudaSuccess) e = cudaStreamWaitEvent(p->s_d2h, p->ev_done[q], 0);
    if (e == cudaSuccess && h_D) e = cudaMemcpyAsync(h_D, f32 ? (void *)p->stageD32[q] : (void *)p->stageD[q], img, cudaMemcpyDeviceToHost, p->s_d2h);
    if (e == cudaSuccess && h_coef)
        e = cudaMemcpyAsync(h_coef, p->stageC[q], (size_t)p->nbatch * p->n * sizeof(double), cudaMemcpyDeviceToHost, p->s_d2h);
    if (e == cudaSuccess) e = cudaEventRecord(p->ev_out[q], p->s_d2h);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return SFFT_OK;
}

int sfft_run_host_async(sfft_plan *p, const double *h_R, const double *h_S, double *h_D, double *h_coef) {
    return run_host_async_any(p, h_R, h_S, h_D, h_coef, false);
}

int sfft_run_host_async_f32(sfft_plan *p, const float *h_R, const float *h_S, float *h_D, double *h_coef) {
    return run_host_async_any(p, h_R, h_S, h_D, h_coef, true);
}

int sfft_run_host_f32(sfft_plan *p, const float *h_R, const float *h_S, float *h_D, double *h_coef) {
    int st = sfft_run_host_async_f32(p, h_R, h_S, h_D, h_coef);
    return st == SFFT_OK ? sfft_run_host_wait(p) : st;
}

int sfft_run_host_wait(sfft_plan *p) {
    if (!p) return SFFT_ERR_INVALID_ARG;
    cudaError_t e = cudaStreamSynchronize(p->s_h2d);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->s_d2h);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return sfft_plan_status(p, nullptr);
}

int sfft_run_host(sfft_plan *p, const double *h_R, const double *h_S, double *h_D, double *h_coef) {
    int st = sfft_run_host_async(p, h_R, h_S, h_D, h_coef);
    return st == SFFT_OK ? sfft_run_host_wait(p) : st;
}

long sfft_plan_launch_count(const sfft_plan *p) { return p ? p->launches : -1; }

void sfft_plan_destroy(sfft_plan *p) {
    if (!p) return;
    for (cudaEvent_t ev : p->prof_events) cudaEventDestroy(ev);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    if (p->side) cudaStreamDestroy(p->side);
    for (int q = 0; q < 2; ++q) {
        if (p->ev_in[q]) cudaEventDestroy(p->ev_in[q]);
        if (p->ev_done[q]) cudaEventDestroy(p->ev_done[q]);
        if (p->ev_out[q]) cudaEventDestroy(p->ev_out[q]);
    }
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    free_tables(p);
    delete p;
}

const char *sfft_strerror(int s) {
    switch (s) {
        case SFFT_OK: return "ok";
        case SFFT_ERR_INVALID_ARG: return "invalid argument";
        case SFFT_ERR_STATE: return "call order violated";
        case SFFT_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
        case SFFT_ERR_CUDA: return "CUDA error (or no CUDA device)";
        case SFFT_ERR_NOT_SPD: return "normal matrix not positive definite";
        default: return "unknown status";
    }
}

const char *sfft_last_cuda_error(const sfft_plan *p) { return p ? p->cuda_err.c_str() : ""; }
const char *sfft_version(void) { return "sfft_b200 0.2 (sm_100a)"; }

}  // extern "C"
