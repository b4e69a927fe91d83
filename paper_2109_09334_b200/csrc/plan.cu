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

void build_jobs(sfft_plan *p) {
    const int FK = p->FK, FB = p->FB, L = p->L, w = p->w, nO = 2 * L - 1;
    p->seqs.clear(); p->jobs.clear(); p->units.clear();
    for (int t = 0; t < FK; ++t) p->seqs.push_back({p->ktj[t], p->kti[t]});
    const int seqS = FK;
    p->seqs.push_back({p->nKa, -1});
    for (int i = 0; i < p->nBa; ++i) p->seqs.push_back({-1, p->nKa + i});
    p->npairs = FK * (FK + 1) / 2;
    p->off_om = 0;
    p->off_th = p->off_om + (size_t)p->npairs * nO * nO;
    p->off_la = p->off_th + (size_t)FK * L * L;
    p->off_de = p->off_la + (size_t)FK * FB * L * L;
    p->tab_size = p->off_de + FB;
    int entry = 0;
    // Omega: kernel terms x kernel terms, lags +-(L-1); only cells with tb <= t are reduced
    for (int a0 = 0; a0 < FK; a0 += kMaxTile)
        for (int b0 = 0; b0 < FK; b0 += kMaxTile) {
            int na = std::min(kMaxTile, FK - a0), nb = std::min(kMaxTile, FK - b0);
            if (b0 + nb - 1 < a0) continue;
            Job j{}; j.na = na; j.nb = nb; j.hw = L - 1; j.out_off = entry;
            for (int q = 0; q < na; ++q) j.a[q] = a0 + q;
            for (int q = 0; q < nb; ++q) j.b[q] = b0 + q;
            for (int ai = 0; ai < na; ++ai)
                for (int bi = 0; bi < nb; ++bi) {
                    int tb = a0 + ai, t = b0 + bi;
                    if (tb > t) continue;
                    for (int r = 0; r < nO; ++r)
                        p->units.push_back({entry + (ai * nb + bi) * nO + r, -1, L - 1,
                                            (int)(p->off_om + ((size_t)pair_index(FK, tb, t) * nO + r) * nO)});
                }
            entry += na * nb * nO;
            p->jobs.push_back(j);
        }
    // Theta (B = S) and Lambda (B = background x-functions), lags +-w
    std::vector<int> bl; bl.push_back(seqS);
    for (int i = 0; i < p->nBa; ++i) bl.push_back(FK + 1 + i);
    for (int a0 = 0; a0 < FK; a0 += kMaxTile)
        for (size_t b0 = 0; b0 < bl.size(); b0 += kMaxTile) {
            int na = std::min(kMaxTile, FK - a0), nb = (int)std::min<size_t>(kMaxTile, bl.size() - b0);
            Job j{}; j.na = na; j.nb = nb; j.hw = w; j.out_off = entry;
            for (int q = 0; q < na; ++q) j.a[q] = a0 + q;
            for (int q = 0; q < nb; ++q) j.b[q] = bl[b0 + q];
            for (int ai = 0; ai < na; ++ai)
                for (int bi = 0; bi < nb; ++bi) {
                    int tb = a0 + ai, sq = j.b[bi];
                    for (int r = 0; r < L; ++r) {
                        int ge = entry + (ai * nb + bi) * L + r;
                        if (sq == seqS) {
                            p->units.push_back({ge, -1, w, (int)(p->off_th + ((size_t)tb * L + r) * L)});
                        } else {
                            int ib = sq - (FK + 1);
                            for (int s = 0; s < FB; ++s)
                                if (p->bti[s] == ib)
                                    p->units.push_back({ge, p->btj[s], w,
                                                        (int)(p->off_la + (((size_t)tb * FB + s) * L + r) * L)});
                        }
                    }
                }
            entry += na * nb * L;
            p->jobs.push_back(j);
        }
    // Delta: A = S, B = background x-functions, lag 0
    for (int b0 = 0; b0 < p->nBa; b0 += kMaxTile) {
        int nb = std::min(kMaxTile, p->nBa - b0);
        Job j{}; j.na = 1; j.nb = nb; j.hw = 0; j.out_off = entry; j.a[0] = seqS;
        for (int q = 0; q < nb; ++q) j.b[q] = FK + 1 + b0 + q;
        for (int bi = 0; bi < nb; ++bi)
            for (int s = 0; s < FB; ++s)
                if (p->bti[s] == b0 + bi) p->units.push_back({entry + bi, p->btj[s], 0, (int)(p->off_de + s)});
        entry += nb;
        p->jobs.push_back(j);
    }
    p->nentries = entry;
}

int fail_cuda(sfft_plan *p, cudaError_t e) {
    if (p) p->cuda_err = cudaGetErrorString(e);
    return SFFT_ERR_CUDA;
}

void free_tables(sfft_plan *p) {
    DeviceTables &d = p->dt;
    cudaFree(d.xwt); cudaFree(d.gK); cudaFree(d.gB); cudaFree(d.twW); cudaFree(d.ghatB); cudaFree(d.phi0);
    cudaFree(d.seqs); cudaFree(d.jobs); cudaFree(d.units);
    cudaFree(d.kti); cudaFree(d.ktj); cudaFree(d.bti); cudaFree(d.btj);
    d = DeviceTables();
}

struct WsLayout {
    size_t rhat, G, tab, M, rhs, Lf, dscale, kfold, ctab, flag, stR, stS, stD, stC, total;
};

WsLayout ws_layout(const sfft_plan *p) {
    WsLayout l{};
    size_t nb = p->nbatch, P = (size_t)p->H * p->W, n = p->n, off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
    l.rhat = take(nb * p->nimg * (size_t)p->H * p->Nh * sizeof(double2));
    l.G = take(nb * (size_t)p->nentries * p->gcols * sizeof(double2));
    l.tab = take(nb * p->tab_size * sizeof(double));
    l.M = take(nb * n * n * sizeof(double));
    l.rhs = take(nb * n * sizeof(double));
    l.Lf = take(nb * (n + 1) * (size_t)p->ldl * sizeof(double));
    l.dscale = take(nb * n * sizeof(double));
    l.kfold = take(nb * (size_t)p->FK * p->L * p->L * sizeof(double));
    l.ctab = take(nb * (size_t)p->H * p->nKa * p->LT * (p->LT + 1) * sizeof(double));
    l.flag = take(nb * sizeof(int) * 2);
    l.stR = take(nb * P * sizeof(double));
    l.stS = take(nb * P * sizeof(double));
    l.stD = take(nb * P * sizeof(double));
    l.stC = take(nb * n * sizeof(double));
    l.total = off;
    return l;
}

}  // namespace

extern "C" {

int sfft_plan_create(sfft_plan **out, int H, int W, int L, int DK, int DB, int basis) {
    if (!out) return SFFT_ERR_INVALID_ARG;
    *out = nullptr;
    if (!is_pow2(H) || !is_pow2(W) || H < 32 || H > 8192 || W < 64 || W > 8192) return SFFT_ERR_INVALID_ARG;
    if (L < 1 || L > 33 || (L % 2) == 0 || 2 * L - 1 > std::min(H, W)) return SFFT_ERR_INVALID_ARG;
    if (DK < 0 || DB < 0 || DK > 8 || DB > 8) return SFFT_ERR_INVALID_ARG;
    if (basis != SFFT_BASIS_POLY && basis != SFFT_BASIS_BSPLINE) return SFFT_ERR_INVALID_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return SFFT_ERR_CUDA; }

    sfft_plan *p = new (std::nothrow) sfft_plan();
    if (!p) return SFFT_ERR_INVALID_ARG;
    p->H = H; p->W = W; p->L = L; p->w = (L - 1) / 2; p->DK = DK; p->DB = DB; p->basis = basis;
    p->Nh = W / 2;
    p->nKa = num_axis(basis, DK); p->nBa = num_axis(basis, DB);
    term_list(basis, DK, p->kti, p->ktj);
    term_list(basis, DB, p->bti, p->btj);
    p->FK = (int)p->kti.size(); p->FB = (int)p->bti.size();
    p->n = p->FK * L * L + p->FB;
    p->nimg = p->nKa + 1;
    p->gcols = p->Nh + 8;
    p->ldl = (p->n + 1 + 7) & ~7;
    p->LT = subtract_tap_width(L);
    build_jobs(p);

    // ---- constant tables (host, long double where it matters) ----
    std::vector<double> fK = axis_table(basis, H, DK), gK = axis_table(basis, W, DK);
    std::vector<double> fB = axis_table(basis, H, DB), gB = axis_table(basis, W, DB);
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
    const int Wh1 = p->Nh + 1;
    std::vector<double2> ghat((size_t)p->nBa * Wh1);
    for (int j = 0; j < p->nBa; ++j)
        for (int m = 0; m < Wh1; ++m) {
            long double re = 0.0L, im = 0.0L;
            for (int y = 0; y < W; ++y) {
                int k = (int)(((long long)m * y) & (W - 1));
                long double g = gB[(size_t)j * W + y];
                re += g * cw[k]; im += g * sw[k];
            }
            ghat[(size_t)j * Wh1 + m] = make_double2((double)re, (double)im);
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

    cudaError_t e = cudaSuccess;
    DeviceTables &d = p->dt;
#define UP(dst, vec) if (e == cudaSuccess) e = upload(&d.dst, vec.data(), vec.size())
    UP(xwt, xwt); UP(gK, gK); UP(gB, gB); UP(twW, twW); UP(ghatB, ghat); UP(phi0, phi0);
    UP(seqs, p->seqs); UP(jobs, p->jobs); UP(units, p->units);
    UP(kti, p->kti); UP(ktj, p->ktj); UP(bti, p->bti); UP(btj, p->btj);
#undef UP
    if (e != cudaSuccess) { free_tables(p); delete p; cudaGetLastError(); return SFFT_ERR_CUDA; }
    *out = p;
    return SFFT_OK;
}

int sfft_plan_set_batch(sfft_plan *p, int nbatch) {
    if (!p || nbatch < 1 || nbatch > 65535) return SFFT_ERR_INVALID_ARG;
    p->nbatch = nbatch; p->ws = nullptr; p->ws_bytes = 0; p->built = p->solved = false;
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
    p->rhat = (double2 *)(b + l.rhat); p->G = (double2 *)(b + l.G); p->tab = (double *)(b + l.tab);
    p->M = (double *)(b + l.M); p->rhs = (double *)(b + l.rhs); p->Lf = (double *)(b + l.Lf);
    p->dscale = (double *)(b + l.dscale); p->kfold = (double *)(b + l.kfold); p->ctab = (double *)(b + l.ctab); p->flag = (int *)(b + l.flag);
    p->stageR = (double *)(b + l.stR); p->stageS = (double *)(b + l.stS); p->stageD = (double *)(b + l.stD);
    p->stageC = (double *)(b + l.stC);
    p->built = p->solved = false;
    return SFFT_OK;
}

int sfft_build_system(sfft_plan *p, const double *d_R, const double *d_S) {
    if (!p || !d_R || !d_S) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    p->built = p->solved = false;
    cudaError_t e = cudaMemsetAsync(p->flag, 0xff, sizeof(int) * 2 * p->nbatch, p->stream);  // -1 = no failure
    if (p->prof_steps > 0) p->prof_cur = p->prof_cur + 1;   // a build opens the next profiled step
    prof_mark(p, 0);
    if (e == cudaSuccess) e = launch_rowfft_forward(p, d_R, d_S);
    prof_mark(p, 1);
    if (e == cudaSuccess) e = launch_corr(p);
    prof_mark(p, 2);
    if (e == cudaSuccess) e = launch_lagsum(p);
    prof_mark(p, 3);
    if (e == cudaSuccess) e = launch_gather(p);
    prof_mark(p, 4);
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
    // stages: 0 rowfft, 1 corr, 2 lagsum, 3 gather, 4 solve, 5 subtract-prep, 6 subtract
    static const int from[SFFT_NUM_STAGES] = {0, 1, 2, 3, 5, 7, 8}, to[SFFT_NUM_STAGES] = {1, 2, 3, 4, 6, 8, 9};
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
    if (ld) *ld = p->n;
    return SFFT_OK;
}

int sfft_get_lag_table(const sfft_plan *p, int which, const double **d_table, size_t *count) {
    if (!p || which < 0 || which > 3) return SFFT_ERR_INVALID_ARG;
    if (!p->built) return SFFT_ERR_STATE;
    if (p->nbatch != 1 && d_table) { /* tables of batch entry b start at b*tab_size; expose entry 0 */ }
    size_t off[5] = {p->off_om, p->off_th, p->off_la, p->off_de, p->tab_size};
    if (d_table) *d_table = p->tab + off[which];
    if (count) *count = off[which + 1] - off[which];
    return SFFT_OK;
}

int sfft_solve(sfft_plan *p, double *d_coef) {
    if (!p || !d_coef) return SFFT_ERR_INVALID_ARG;
    if (!p->built) return SFFT_ERR_STATE;
    prof_mark(p, 5);
    cudaError_t e = launch_solve(p, d_coef);
    prof_mark(p, 6);
    if (e != cudaSuccess) return fail_cuda(p, e);
    p->solved = true;
    return SFFT_OK;
}

int sfft_subtract(sfft_plan *p, const double *d_coef, const double *d_R, const double *d_S, double *d_D) {
    if (!p || !d_coef || !d_R || !d_S || !d_D) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    prof_mark(p, 7);
    cudaError_t e = launch_subtract(p, d_coef, d_R, d_S, d_D);
    prof_mark(p, 9);
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
            if (info) *info = b * p->n + h[2 * b];
            return SFFT_ERR_NOT_SPD;
        }
    return SFFT_OK;
}

int sfft_run_host(sfft_plan *p, const double *h_R, const double *h_S, double *h_D, double *h_coef) {
    if (!p || !h_R || !h_S) return SFFT_ERR_INVALID_ARG;
    if (!p->ws) return SFFT_ERR_WORKSPACE;
    size_t img = (size_t)p->nbatch * p->H * p->W * sizeof(double);
    cudaError_t e = cudaMemcpyAsync(p->stageR, h_R, img, cudaMemcpyHostToDevice, p->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(p->stageS, h_S, img, cudaMemcpyHostToDevice, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e);
    int st = sfft_build_system(p, p->stageR, p->stageS);
    if (st == SFFT_OK) st = sfft_solve(p, p->stageC);
    if (st == SFFT_OK) st = sfft_subtract(p, p->stageC, p->stageR, p->stageS, p->stageD);
    if (st != SFFT_OK) return st;
    if (h_D) e = cudaMemcpyAsync(h_D, p->stageD, img, cudaMemcpyDeviceToHost, p->stream);
    if (e == cudaSuccess && h_coef)
        e = cudaMemcpyAsync(h_coef, p->stageC, (size_t)p->nbatch * p->n * sizeof(double), cudaMemcpyDeviceToHost, p->stream);
    if (e != cudaSuccess) return fail_cuda(p, e);
    return sfft_plan_status(p, nullptr);
}

long sfft_plan_launch_count(const sfft_plan *p) { return p ? p->launches : -1; }

void sfft_plan_destroy(sfft_plan *p) {
    if (!p) return;
    for (cudaEvent_t ev : p->prof_events) cudaEventDestroy(ev);
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
const char *sfft_version(void) { return "sfft_b200 0.1 (sm_100a)"; }

}  // extern "C"
