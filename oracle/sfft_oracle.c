/*
 * sfft_oracle.c -- CPU ORACLE for the SFFT hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code with the CUDA path (paper_2109_09334_b200/csrc)
 * and uses NO FFT anywhere: every quantity is the plain real-space definition written
 * out as loops, in FP64 with long-double combination of partial sums.
 *
 * What it computes (citations are PAPER.md line + equation; "DESIGN g#" = a reading
 * of a garbled/silent passage listed in DESIGN.md):
 *
 *   D(x,y) = S(x,y) - sum_{t,ab} a_{t,ab} (R^t o K_ab)(x,y) - sum_s b_s T'_s(x,y)   (Eq. 12)
 *   K_00 = delta,  K_ab = delta(u-a,v-b) - delta(u,v)                               (Eqs. 3-4)
 *   R^t = T_t * R  (weights inside the circular convolution)                        (Eq. 11)
 *   T_t : monomials of normalised coordinates (Eqs. 2, 6; DESIGN g8) or
 *         tensor-product cubic B-splines (Eqs. 8-9; DESIGN g13)
 *   least squares over all pixels  ==  the paper's Fourier-space minimisation by
 *   Parseval (Eqs. 15-18), so  M = Phi^T Phi,  rhs = Phi^T S.
 *
 * Two tiers for the normal system:
 *   Tier A  orc_design_matrix + orc_gram : materialise Phi (P x n) and take every dot
 *           product from the definition.  Tiny inputs only (n^2 P / 2 work).
 *   Tier B  orc_lag_tables + orc_gather  : the lag form of App. B
 *           with every correlation evaluated as a DIRECT PIXEL SUM, in the
 *           cancellation-free form  Q(rho) = sum_x A(x) [B(x+rho) - B(x)].
 *           Tier B is pinned to Tier A in tests/test_oracle_pins.py.
 *
 * Index conventions (shared with include/sfft.h by specification, not by code):
 *   arrays row-major [x][y], x in [0,H) slow, y in [0,W) fast;  P = H*W;  L = 2w+1
 *   lag index   a = (alpha+w)*L + (beta+w),  centre a0 = w*L + w
 *   unknown     k = t*L*L + a  (kernel),  k = F_K*L*L + s  (background);  n = F_K*L*L + F_B
 *   POLY terms  t <-> (i,j): i = 0..D outer, j = 0..D-i inner, T_t = u_x^i u_y^j
 *   BSPLINE     t = i*nb + j, nb = m+4, T_t = B_i(v_x) B_j(v_y)
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_POLY 0
#define ORC_BSPLINE 1

/* ---------------------------------------------------------------- weights */

/* number of 1-D functions per axis, and of 2-D terms */
int orc_num_axis(int basis, int D) { return basis == ORC_POLY ? D + 1 : D + 4; }
int orc_num_terms(int basis, int D) {
    return basis == ORC_POLY ? (D + 1) * (D + 2) / 2 : (D + 4) * (D + 4);
}

/* term list t -> (i,j).  POLY: PAPER.md:86,105 index ranges.  BSPLINE: Eqs. 8-9 sum over all i,j. */
void orc_terms(int basis, int D, int *ti, int *tj) {
    int t = 0;
    if (basis == ORC_POLY) {
        for (int i = 0; i <= D; ++i)
            for (int j = 0; j <= D - i; ++j) { ti[t] = i; tj[t] = j; ++t; }
    } else {
        int nb = D + 4;
        for (int i = 0; i < nb; ++i)
            for (int j = 0; j < nb; ++j) { ti[t] = i; tj[t] = j; ++t; }
    }
}

/* Cox-de Boor recursion, degree k, knot vector tk[], half-open intervals (DESIGN g13). */
static long double bspline_cdb(int i, int k, const long double *tk, long double v) {
    if (k == 0) return (tk[i] <= v && v < tk[i + 1]) ? 1.0L : 0.0L;
    long double a = 0.0L, b = 0.0L;
    long double d1 = tk[i + k] - tk[i], d2 = tk[i + k + 1] - tk[i + 1];
    if (d1 > 0.0L) a = (v - tk[i]) / d1 * bspline_cdb(i, k - 1, tk, v);
    if (d2 > 0.0L) b = (tk[i + k + 1] - v) / d2 * bspline_cdb(i + 1, k - 1, tk, v);
    return a + b;
}

/* 1-D basis table out[f][x], f < orc_num_axis, x < N.
 * POLY   : u = (2x+1)/N - 1 in (-1,1),  out[f][x] = u^f                      (DESIGN g8)
 * BSPLINE: v = (x+0.5)/N in (0,1), cubic, clamped knots with D uniform interior knots. */
void orc_axis_table(int basis, int N, int D, double *out) {
    if (basis == ORC_POLY) {
        for (int x = 0; x < N; ++x) {
            long double u = (2.0L * x + 1.0L) / N - 1.0L, p = 1.0L;
            for (int f = 0; f <= D; ++f) { out[(size_t)f * N + x] = (double)p; p *= u; }
        }
    } else {
        int m = D, nb = m + 4, nk = m + 8;
        long double *tk = (long double *)malloc(sizeof(long double) * nk);
        for (int q = 0; q < 4; ++q) { tk[q] = 0.0L; tk[nk - 1 - q] = 1.0L; }
        for (int q = 1; q <= m; ++q) tk[3 + q] = (long double)q / (m + 1);
        for (int x = 0; x < N; ++x) {
            long double v = (x + 0.5L) / N;
            for (int f = 0; f < nb; ++f) out[(size_t)f * N + x] = (double)bspline_cdb(f, 3, tk, v);
        }
        free(tk);
    }
}

/* weighted image out(x,y) = f_i(x) g_j(y) img(x,y); img==NULL means img = 1 (gives T_t itself) */
static void weighted_image(int H, int W, const double *fx, const double *gy, const double *img, double *out) {
    for (int x = 0; x < H; ++x)
        for (int y = 0; y < W; ++y)
            out[(size_t)x * W + y] = fx[x] * gy[y] * (img ? img[(size_t)x * W + y] : 1.0);
}

typedef struct {
    int FK, FB, nKa, nBa;
    int *kti, *ktj, *bti, *btj;
    double *fK, *gK, *fB, *gB; /* axis tables: kernel x [nKa][H], kernel y [nKa][W], bg x, bg y */
} orc_basis;

static void basis_make(orc_basis *b, int H, int W, int basis, int DK, int DB) {
    b->FK = orc_num_terms(basis, DK); b->FB = orc_num_terms(basis, DB);
    b->nKa = orc_num_axis(basis, DK); b->nBa = orc_num_axis(basis, DB);
    b->kti = (int *)malloc(sizeof(int) * b->FK); b->ktj = (int *)malloc(sizeof(int) * b->FK);
    b->bti = (int *)malloc(sizeof(int) * b->FB); b->btj = (int *)malloc(sizeof(int) * b->FB);
    orc_terms(basis, DK, b->kti, b->ktj); orc_terms(basis, DB, b->bti, b->btj);
    b->fK = (double *)malloc(sizeof(double) * b->nKa * H); b->gK = (double *)malloc(sizeof(double) * b->nKa * W);
    b->fB = (double *)malloc(sizeof(double) * b->nBa * H); b->gB = (double *)malloc(sizeof(double) * b->nBa * W);
    orc_axis_table(basis, H, DK, b->fK); orc_axis_table(basis, W, DK, b->gK);
    orc_axis_table(basis, H, DB, b->fB); orc_axis_table(basis, W, DB, b->gB);
}
static void basis_free(orc_basis *b) {
    free(b->kti); free(b->ktj); free(b->bti); free(b->btj);
    free(b->fK); free(b->gK); free(b->fB); free(b->gB);
}

int orc_num_unknowns(int L, int basis, int DK, int DB) {
    return orc_num_terms(basis, DK) * L * L + orc_num_terms(basis, DB);
}

static inline int wrap(int v, int N) { v %= N; return v < 0 ? v + N : v; }

/* ---------------------------------------------------------------- Tier A */

/* Phi[k][p], k < n, p = x*W+y.  Column k of the design matrix (Eqs. 3-4, 11-12):
 *   kernel unknown (t, a=(alpha,beta)):  V = R^t shifted by (alpha,beta) circularly,
 *                                        minus R^t itself unless (alpha,beta)=(0,0)
 *   background unknown s:                T'_s                                          */
void orc_design_matrix(int H, int W, int L, int basis, int DK, int DB, const double *R, double *Phi) {
    orc_basis b; basis_make(&b, H, W, basis, DK, DB);
    int w = (L - 1) / 2; size_t P = (size_t)H * W;
    double *Rt = (double *)malloc(sizeof(double) * P);
    for (int t = 0; t < b.FK; ++t) {
        weighted_image(H, W, b.fK + (size_t)b.kti[t] * H, b.gK + (size_t)b.ktj[t] * W, R, Rt);
        for (int al = -w; al <= w; ++al)
            for (int be = -w; be <= w; ++be) {
                int a = (al + w) * L + (be + w);
                double *col = Phi + ((size_t)t * L * L + a) * P;
                int centre = (al == 0 && be == 0);
                for (int x = 0; x < H; ++x)
                    for (int y = 0; y < W; ++y) {
                        double sh = Rt[(size_t)wrap(x - al, H) * W + wrap(y - be, W)];
                        col[(size_t)x * W + y] = centre ? sh : sh - Rt[(size_t)x * W + y];
                    }
            }
    }
    for (int s = 0; s < b.FB; ++s)
        weighted_image(H, W, b.fB + (size_t)b.bti[s] * H, b.gB + (size_t)b.btj[s] * W, NULL,
                       Phi + ((size_t)b.FK * L * L + s) * P);
    free(Rt); basis_free(&b);
}

/* M = Phi^T Phi (full symmetric, both triangles written), rhs = Phi^T S; long-double sums. */
void orc_gram(int n, long P, const double *Phi, const double *S, double *M, double *rhs) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n; ++k) {
        const double *ck = Phi + (size_t)k * P;
        for (int k2 = 0; k2 <= k; ++k2) {
            const double *c2 = Phi + (size_t)k2 * P;
            long double acc = 0.0L;
            for (long p = 0; p < P; ++p) acc += (long double)ck[p] * c2[p];
            M[(size_t)k * n + k2] = M[(size_t)k2 * n + k] = (double)acc;
        }
        long double acc = 0.0L;
        for (long p = 0; p < P; ++p) acc += (long double)ck[p] * S[p];
        rhs[k] = (double)acc;
    }
}

/* diag[k] = sum_p Phi_k(p)^2 and rhs[k] = sum_p Phi_k(p) S(p) for every unknown k, straight from the column
 * definitions of orc_design_matrix (Eqs. 3-4, 11-12) without materialising Phi: the diagonal of the normal
 * matrix and the whole right-hand side at 2 n P multiply-adds, cheap enough to check every entry of a large
 * batch (config 5: all 64 sub-fields).  Row partial sums in double, rows combined in long double. */
void orc_diag_and_rhs(int H, int W, int L, int basis, int DK, int DB, const double *R, const double *S,
                      double *diag, double *rhs) {
    orc_basis b; basis_make(&b, H, W, basis, DK, DB);
    int w = (L - 1) / 2, LL = L * L; size_t P = (size_t)H * W;
    double *Rt = (double *)malloc(sizeof(double) * P);
    for (int t = 0; t < b.FK; ++t) {
        weighted_image(H, W, b.fK + (size_t)b.kti[t] * H, b.gK + (size_t)b.ktj[t] * W, R, Rt);
        /* rows outermost (each image row is read once per term), all L*L lags per row; per-thread long-double
         * accumulators of double row partial sums, combined at the end */
        long double *acc2 = (long double *)calloc((size_t)LL, sizeof(long double));
        long double *accs = (long double *)calloc((size_t)LL, sizeof(long double));
#pragma omp parallel
        {
            long double *l2 = (long double *)calloc((size_t)LL, sizeof(long double));
            long double *ls = (long double *)calloc((size_t)LL, sizeof(long double));
            double *sh = (double *)malloc(sizeof(double) * W);       /* sh[y] = R^t((x-al)%H, (y-be)%W) */
#pragma omp for schedule(static)
            for (int x = 0; x < H; ++x) {
                const double *own = Rt + (size_t)x * W, *sr = S + (size_t)x * W;
                for (int a = 0; a < LL; ++a) {
                    int al = a / L - w, be = a % L - w, centre = (al == 0 && be == 0);
                    const double *src = Rt + (size_t)wrap(x - al, H) * W;
                    int o = wrap(-be, W);                     /* sh[y] = src[(y + o) % W], in two runs */
                    for (int y = 0; y < W - o; ++y) sh[y] = src[y + o];
                    for (int y = W - o; y < W; ++y) sh[y] = src[y + o - W];
                    double r2 = 0.0, rs = 0.0, cm = centre ? 0.0 : 1.0;
#pragma omp simd reduction(+ : r2, rs)
                    for (int y = 0; y < W; ++y) {
                        double v = sh[y] - cm * own[y];
                        r2 += v * v; rs += v * sr[y];
                    }
                    l2[a] += r2; ls[a] += rs;
                }
            }
#pragma omp critical
            for (int a = 0; a < LL; ++a) { acc2[a] += l2[a]; accs[a] += ls[a]; }
            free(l2); free(ls); free(sh);
        }
        for (int a = 0; a < LL; ++a) { diag[(size_t)t * LL + a] = (double)acc2[a]; rhs[(size_t)t * LL + a] = (double)accs[a]; }
        free(acc2); free(accs);
    }
    for (int s = 0; s < b.FB; ++s) {
        const double *fx = b.fB + (size_t)b.bti[s] * H, *gy = b.gB + (size_t)b.btj[s] * W;
        long double a2 = 0.0L, as = 0.0L;
        for (int x = 0; x < H; ++x) {
            double r2 = 0.0, rs = 0.0;
            for (int y = 0; y < W; ++y) { double v = fx[x] * gy[y]; r2 += v * v; rs += v * S[(size_t)x * W + y]; }
            a2 += r2; as += rs;
        }
        diag[(size_t)b.FK * LL + s] = (double)a2; rhs[(size_t)b.FK * LL + s] = (double)as;
    }
    free(Rt); basis_free(&b);
}

/* ---------------------------------------------------------------- Tier B */

/* Direct-sum correlation in difference form, all lags |rho|,|eps| <= wl:
 *   q[(rho+wl)*(2wl+1) + (eps+wl)] = sum_{x,y} A(x,y) * ( B((x+rho)%H,(y+eps)%W) - B(x,y) )
 *   *c0 = sum_{x,y} A(x,y) B(x,y)
 * so that the paper's correlation array (App. B) is Omega(rho,eps) = q + c0.
 * Row partial sums in double, rows combined in long double. */
static void corr_diff(int H, int W, const double *A, const double *B, int wl, double *q, double *c0) {
    int nl = 2 * wl + 1;
    long double *acc = (long double *)calloc((size_t)nl * nl + 1, sizeof(long double));
#pragma omp parallel
    {
        long double *loc = (long double *)calloc((size_t)nl * nl + 1, sizeof(long double));
        double *Bp = (double *)malloc(sizeof(double) * (W + 2 * wl)); /* wrapped copy of the shifted row */
#pragma omp for schedule(static)
        for (int x = 0; x < H; ++x) {
            const double *a = A + (size_t)x * W, *b0 = B + (size_t)x * W;
            double s0 = 0.0;
            for (int y = 0; y < W; ++y) s0 += a[y] * b0[y];
            loc[(size_t)nl * nl] += s0;
            for (int rho = -wl; rho <= wl; ++rho) {
                const double *b1 = B + (size_t)wrap(x + rho, H) * W;
                for (int y = -wl; y < W + wl; ++y) Bp[y + wl] = b1[wrap(y, W)];
                for (int eps = -wl; eps <= wl; ++eps) {
                    const double *bs = Bp + wl + eps;
                    double s = 0.0;
                    for (int y = 0; y < W; ++y) s += a[y] * (bs[y] - b0[y]);
                    loc[(size_t)(rho + wl) * nl + (eps + wl)] += s;
                }
            }
        }
#pragma omp critical
        for (size_t i = 0; i < (size_t)nl * nl + 1; ++i) acc[i] += loc[i];
        free(loc); free(Bp);
    }
    for (size_t i = 0; i < (size_t)nl * nl; ++i) q[i] = (double)acc[i];
    *c0 = (double)acc[(size_t)nl * nl];
    free(acc);
}

/* one lag only (used for sampled full-size checks): returns q(rho,eps) and c0 via pointer */
double orc_corr_diff_one(int H, int W, const double *A, const double *B, int rho, int eps, double *c0) {
    long double acc = 0.0L, acc0 = 0.0L;
#pragma omp parallel for reduction(+ : acc, acc0) schedule(static)
    for (int x = 0; x < H; ++x) {
        const double *a = A + (size_t)x * W, *b0 = B + (size_t)x * W, *b1 = B + (size_t)wrap(x + rho, H) * W;
        double s = 0.0, s0 = 0.0;
        for (int y = 0; y < W; ++y) { s += a[y] * (b1[wrap(y + eps, W)] - b0[y]); s0 += a[y] * b0[y]; }
        acc += s; acc0 += s0;
    }
    if (c0) *c0 = (double)acc0;
    return (double)acc;
}

/* weighted reference image R^t for term t (exported for sampled checks) */
void orc_weighted_ref(int H, int W, int basis, int DK, int t, const double *R, double *out) {
    orc_basis b; basis_make(&b, H, W, basis, DK, 0);
    weighted_image(H, W, b.fK + (size_t)b.kti[t] * H, b.gK + (size_t)b.ktj[t] * W, R, out);
    basis_free(&b);
}

/* Lag tables by direct pixel sums (no FFT).  Layout (nO = 2L-1, wl = L-1 for Omega; L, w for the others):
 *   Qom [FK][FK][nO][nO]  only tb <= t filled:  Omega_{tb,t}(rho,eps) - Omega_{tb,t}(0,0),
 *                         Omega_{tb,t}(rho,eps) = sum R^tb(x,y) R^t(x+rho,y+eps)        (B6, DESIGN g2)
 *   Om0 [FK][FK]          Omega_{tb,t}(0,0)   (tb <= t)
 *   Qla [FK][FB][L][L]    Lambda_{tb,s}(rho,eps) - Lambda_{tb,s}(0,0),  Lambda = sum R^tb(x) T'_s(x+rho)   (B8)
 *   La0 [FK][FB]
 *   Qth [FK][L][L]        Theta_tb(rho,eps) - Theta_tb(0,0),  Theta = sum R^tb(x) S(x+rho)   (B14, DESIGN g2)
 *   Th0 [FK]
 *   Phi0[FB][FB]          sum T'_sb T'_s    (B11/B12 at lag 0)
 *   De0 [FB]              sum S T'_s        (B15/B16 at lag 0)                                             */
void orc_lag_tables(int H, int W, int L, int basis, int DK, int DB, const double *R, const double *S,
                    double *Qom, double *Om0, double *Qla, double *La0, double *Qth, double *Th0,
                    double *Phi0, double *De0) {
    orc_basis b; basis_make(&b, H, W, basis, DK, DB);
    int w = (L - 1) / 2, nO = 2 * L - 1; size_t P = (size_t)H * W;
    int FK = b.FK, FB = b.FB;
    double *Rt = (double *)malloc(sizeof(double) * P * FK);
    double *Ts = (double *)malloc(sizeof(double) * P * FB);
    for (int t = 0; t < FK; ++t)
        weighted_image(H, W, b.fK + (size_t)b.kti[t] * H, b.gK + (size_t)b.ktj[t] * W, R, Rt + P * t);
    for (int s = 0; s < FB; ++s)
        weighted_image(H, W, b.fB + (size_t)b.bti[s] * H, b.gB + (size_t)b.btj[s] * W, NULL, Ts + P * s);
    for (int tb = 0; tb < FK; ++tb) {
        for (int t = tb; t < FK; ++t)
            corr_diff(H, W, Rt + P * tb, Rt + P * t, L - 1, Qom + ((size_t)tb * FK + t) * nO * nO, Om0 + tb * FK + t);
        for (int s = 0; s < FB; ++s)
            corr_diff(H, W, Rt + P * tb, Ts + P * s, w, Qla + ((size_t)tb * FB + s) * L * L, La0 + tb * FB + s);
        corr_diff(H, W, Rt + P * tb, S, w, Qth + (size_t)tb * L * L, Th0 + tb);
    }
    for (int sb = 0; sb < FB; ++sb) {
        for (int s = 0; s < FB; ++s) {
            long double acc = 0.0L;
            for (size_t p = 0; p < P; ++p) acc += (long double)Ts[P * sb + p] * Ts[P * s + p];
            Phi0[sb * FB + s] = (double)acc;
        }
        long double acc = 0.0L;
        for (size_t p = 0; p < P; ++p) acc += (long double)S[p] * Ts[P * sb + p];
        De0[sb] = (double)acc;
    }
    free(Rt); free(Ts); basis_free(&b);
}

/* Assemble M (n x n, full symmetric) and rhs from the lag tables: App. B in real-space scaling.
 *   (B5, missing from PAPER.md:505-507; reading DESIGN g1)  with Q = Omega - Omega(0,0):
 *     both lags != 0 : Omega(ab-a) - Omega(ab) - Omega(-a) + Omega(0) = Q(ab-a) - Q(ab) - Q(-a)
 *     only a  = 0    : Omega(ab) - Omega(0)  = Q(ab)
 *     only ab = 0    : Omega(-a) - Omega(0)  = Q(-a)
 *     both 0         : Omega(0)
 *   (B7)  M_ab = Lambda(ab) - Lambda(0)  | Lambda(0) at the centre
 *   (B9)  M_ba = M_ab^T                                                (DESIGN g5)
 *   (B11) M_bb = Phi(0,0)
 *   (B13) rhs_a = Theta(ab) - Theta(0) | Theta(0) at the centre
 *   (B15) rhs_b = Delta(0,0)
 *   For tb > t:  Omega_{tb,t}(rho) = Omega_{t,tb}(-rho).                                     */
void orc_gather(int L, int FK, int FB, const double *Qom, const double *Om0, const double *Qla,
                const double *La0, const double *Qth, const double *Th0, const double *Phi0,
                const double *De0, double *M, double *rhs) {
    int w = (L - 1) / 2, nO = 2 * L - 1, LL = L * L, n = FK * LL + FB, wl = L - 1;
#define QOM(tb, t, r, e)                                                              \
    ((tb) <= (t) ? Qom[(((size_t)(tb)*FK + (t)) * nO + ((r) + wl)) * nO + ((e) + wl)] \
                 : Qom[(((size_t)(t)*FK + (tb)) * nO + (-(r) + wl)) * nO + (-(e) + wl)])
#define OM0(tb, t) ((tb) <= (t) ? Om0[(tb)*FK + (t)] : Om0[(t)*FK + (tb)])
    for (int tb = 0; tb < FK; ++tb)
        for (int alb = -w; alb <= w; ++alb)
            for (int beb = -w; beb <= w; ++beb) {
                int kb = tb * LL + (alb + w) * L + (beb + w);
                int cb = (alb == 0 && beb == 0);
                for (int t = 0; t < FK; ++t)
                    for (int al = -w; al <= w; ++al)
                        for (int be = -w; be <= w; ++be) {
                            int k = t * LL + (al + w) * L + (be + w);
                            int c = (al == 0 && be == 0);
                            double v;
                            if (cb && c) v = OM0(tb, t);
                            else if (c) v = QOM(tb, t, alb, beb);
                            else if (cb) v = QOM(tb, t, -al, -be);
                            else v = QOM(tb, t, alb - al, beb - be) - QOM(tb, t, alb, beb) - QOM(tb, t, -al, -be);
                            if (kb <= k) M[(size_t)kb * n + k] = M[(size_t)k * n + kb] = v; /* M = M^T by definition */
                        }
                for (int s = 0; s < FB; ++s) {
                    double v = cb ? La0[tb * FB + s] : Qla[((size_t)(tb * FB + s) * L + (alb + w)) * L + (beb + w)];
                    M[(size_t)kb * n + FK * LL + s] = v;
                    M[(size_t)(FK * LL + s) * n + kb] = v;
                }
                rhs[kb] = cb ? Th0[tb] : Qth[((size_t)tb * L + (alb + w)) * L + (beb + w)];
            }
    for (int sb = 0; sb < FB; ++sb) {
        for (int s = 0; s < FB; ++s) M[(size_t)(FK * LL + sb) * n + FK * LL + s] = Phi0[sb * FB + s];
        rhs[FK * LL + sb] = De0[sb];
    }
#undef QOM
#undef OM0
}

/* ---------------------------------------------------------------- solve */

/* Solve M c = rhs for SPD M (DESIGN g11): Jacobi scaling, unblocked Cholesky, two triangular
 * solves, then `refine` steps of iterative refinement with a long-double residual.
 * Returns 0, or k+1 if pivot k is not positive (M not SPD).  M is not modified. */
int orc_solve(int n, const double *M, const double *rhs, double *c, int refine) {
    double *Lm = (double *)malloc(sizeof(double) * (size_t)n * n);
    double *d = (double *)malloc(sizeof(double) * n), *r = (double *)malloc(sizeof(double) * n);
    double *z = (double *)malloc(sizeof(double) * n);
    int info = 0;
    for (int i = 0; i < n; ++i) {
        if (!(M[(size_t)i * n + i] > 0.0)) { info = i + 1; goto done; }
        d[i] = 1.0 / sqrt(M[(size_t)i * n + i]);
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) Lm[(size_t)i * n + j] = M[(size_t)i * n + j] * d[i] * d[j];
    /* Cholesky, row-oriented (Cholesky-Banachiewicz): L[i][j] = (A[i][j] - sum_k L[i][k] L[j][k]) / L[j][j] */
    for (int j = 0; j < n; ++j) {
        long double s = Lm[(size_t)j * n + j];
        for (int k = 0; k < j; ++k) s -= (long double)Lm[(size_t)j * n + k] * Lm[(size_t)j * n + k];
        if (!(s > 0.0L)) { info = j + 1; goto done; }
        double ljj = sqrt((double)s);
        Lm[(size_t)j * n + j] = ljj;
#pragma omp parallel for schedule(static) if (n - j > 256)
        for (int i = j + 1; i < n; ++i) {
            double t = Lm[(size_t)i * n + j];
            const double *li = Lm + (size_t)i * n, *lj = Lm + (size_t)j * n;
            double acc = 0.0;
            for (int k = 0; k < j; ++k) acc += li[k] * lj[k];
            Lm[(size_t)i * n + j] = (t - acc) / ljj;
        }
    }
    for (int i = 0; i < n; ++i) c[i] = 0.0;
    for (int it = 0; it <= refine; ++it) {
        /* residual of the ORIGINAL system in long double, then scaled: r = D (rhs - M c) */
#pragma omp parallel for schedule(static)
        for (int i = 0; i < n; ++i) {
            long double acc = rhs[i];
            for (int j = 0; j < n; ++j) acc -= (long double)M[(size_t)i * n + j] * c[j];
            r[i] = (double)(acc * d[i]);
        }
        for (int i = 0; i < n; ++i) { /* L z = r */
            long double acc = r[i];
            for (int k = 0; k < i; ++k) acc -= (long double)Lm[(size_t)i * n + k] * z[k];
            z[i] = (double)(acc / Lm[(size_t)i * n + i]);
        }
        for (int i = n - 1; i >= 0; --i) { /* L^T y = z */
            long double acc = z[i];
            for (int k = i + 1; k < n; ++k) acc -= (long double)Lm[(size_t)k * n + i] * z[k];
            z[i] = (double)(acc / Lm[(size_t)i * n + i]);
        }
        for (int i = 0; i < n; ++i) c[i] += z[i] * d[i];
    }
done:
    free(Lm); free(d); free(r); free(z);
    return info;
}

/* ---------------------------------------------------------------- difference */

/* D = S - sum_t sum_ab k_{t,ab} R^t((x-a)%H,(y-b)%W) - sum_s b_s T'_s        (Eqs. 1, 12)
 * with k_{t,ab} = a_{t,ab} for (a,b) != 0 and k_{t,00} = a_{t,00} - sum_{ab != 0} a_{t,ab}  (Eqs. 3-4).
 * (R,S) may differ from the fitted pair. */
void orc_difference(int H, int W, int L, int basis, int DK, int DB, const double *R, const double *S,
                    const double *c, double *D) {
    orc_basis b; basis_make(&b, H, W, basis, DK, DB);
    int w = (L - 1) / 2, LL = L * L, FK = b.FK, FB = b.FB; size_t P = (size_t)H * W;
    double *kk = (double *)malloc(sizeof(double) * FK * LL);
    for (int t = 0; t < FK; ++t) {
        long double s = 0.0L;
        for (int a = 0; a < LL; ++a) { kk[t * LL + a] = c[t * LL + a]; if (a != w * L + w) s += c[t * LL + a]; }
        kk[t * LL + w * L + w] = (double)((long double)c[t * LL + w * L + w] - s);
    }
    double *Rt = (double *)malloc(sizeof(double) * P * FK);
    for (int t = 0; t < FK; ++t)
        weighted_image(H, W, b.fK + (size_t)b.kti[t] * H, b.gK + (size_t)b.ktj[t] * W, R, Rt + P * t);
#pragma omp parallel for schedule(static)
    for (int x = 0; x < H; ++x)
        for (int y = 0; y < W; ++y) {
            long double acc = S[(size_t)x * W + y];
            for (int t = 0; t < FK; ++t) {
                const double *im = Rt + P * t, *kt = kk + t * LL;
                for (int al = -w; al <= w; ++al) {
                    const double *row = im + (size_t)wrap(x - al, H) * W;
                    double part = 0.0;
                    for (int be = -w; be <= w; ++be) part += kt[(al + w) * L + (be + w)] * row[wrap(y - be, W)];
                    acc -= part;
                }
            }
            for (int s = 0; s < FB; ++s)
                acc -= (long double)c[FK * LL + s] * b.fB[(size_t)b.bti[s] * H + x] * b.gB[(size_t)b.btj[s] * W + y];
            D[(size_t)x * W + y] = (double)acc;
        }
    free(kk); free(Rt); basis_free(&b);
}

/* D at selected pixels only (full-size sampled checks); px,py arrays of length npix */
void orc_difference_at(int H, int W, int L, int basis, int DK, int DB, const double *R, const double *S,
                       const double *c, int npix, const int *px, const int *py, double *Dout) {
    orc_basis b; basis_make(&b, H, W, basis, DK, DB);
    int w = (L - 1) / 2, LL = L * L, FK = b.FK, FB = b.FB;
    for (int q = 0; q < npix; ++q) {
        int x = px[q], y = py[q];
        long double acc = S[(size_t)x * W + y];
        for (int t = 0; t < FK; ++t) {
            const double *fx = b.fK + (size_t)b.kti[t] * H, *gy = b.gK + (size_t)b.ktj[t] * W;
            long double centre = 0.0L;
            for (int al = -w; al <= w; ++al)
                for (int be = -w; be <= w; ++be) {
                    int xs = wrap(x - al, H), ys = wrap(y - be, W);
                    double rt = fx[xs] * gy[ys] * R[(size_t)xs * W + ys];
                    double a = c[t * LL + (al + w) * L + (be + w)];
                    if (al == 0 && be == 0) acc -= (long double)a * rt;
                    else { acc -= (long double)a * rt; centre += a; }
                }
            acc += centre * (long double)(fx[x] * gy[y] * R[(size_t)x * W + y]);
        }
        for (int s = 0; s < FB; ++s)
            acc -= (long double)c[FK * LL + s] * b.fB[(size_t)b.bti[s] * H + x] * b.gB[(size_t)b.btj[s] * W + y];
        Dout[q] = (double)acc;
    }
    basis_free(&b);
}

/* ---------------------------------------------------------------------------------------------
 * NEXT-1: constant photometric ratio.  "The constant flux scaling between
 * images requires a constant kernel integral, that is, A_xy00 = a_0000": the kernel-sum field
 * sum_t a_{t,00} T_t(x,y) must not depend on position.
 *   POLY    : T_0 = 1 and the other monomials vary  =>  a_{t,00} = 0 for t >= 1.
 *   BSPLINE : the T_t form a partition of unity      =>  all a_{t,00} equal.
 * Either way c = C c' with one shared unknown s in place of the F_K centre coefficients:
 *   c_k = c'_{r(k)} for a non-centre k;  c_{t*LL+a0} = omega_t * c'_s,  omega = e_0 (POLY) or 1 (BSPLINE),
 * and the basis image of s is sum_t omega_t R^t = R.  The reduced unknowns keep the original order with
 * the centre entries of t >= 1 removed (s sits where a_{0,00} was), n' = n - (F_K - 1).
 * Least squares over c' has the normal system  M' = C^T M C,  rhs' = C^T rhs  (plain definition).
 * ------------------------------------------------------------------------------------------- */
int orc_cpr_num_unknowns(int L, int basis, int DK, int DB) {
    return orc_num_unknowns(L, basis, DK, DB) - (orc_num_terms(basis, DK) - 1);
}

/* map[k] = reduced index of full unknown k; wgt[k] = its weight omega (1 for non-centre entries) */
static void cpr_map(int L, int basis, int DK, int DB, int *map, double *wgt) {
    int FK = orc_num_terms(basis, DK), LL = L * L, a0 = (L / 2) * L + L / 2, n = orc_num_unknowns(L, basis, DK, DB);
    int next = 0;
    for (int k = 0; k < n; ++k) {
        int centre = (k < FK * LL) && (k % LL == a0), t = k / LL;
        if (centre && t >= 1) { map[k] = a0; wgt[k] = (basis == ORC_POLY) ? 0.0 : 1.0; }
        else { map[k] = next++; wgt[k] = 1.0; }
    }
}

void orc_cpr_constrain(int L, int basis, int DK, int DB, const double *M, const double *rhs, double *Mc, double *rc) {
    int n = orc_num_unknowns(L, basis, DK, DB), nr = orc_cpr_num_unknowns(L, basis, DK, DB);
    int *map = (int *)malloc(sizeof(int) * n);
    double *wgt = (double *)malloc(sizeof(double) * n);
    long double *acc = (long double *)calloc((size_t)nr * nr, sizeof(long double));
    long double *ar = (long double *)calloc((size_t)nr, sizeof(long double));
    cpr_map(L, basis, DK, DB, map, wgt);
    for (int k = 0; k < n; ++k) {
        ar[map[k]] += (long double)wgt[k] * rhs[k];
        for (int l = 0; l < n; ++l) acc[(size_t)map[k] * nr + map[l]] += (long double)wgt[k] * wgt[l] * M[(size_t)k * n + l];
    }
    for (size_t i = 0; i < (size_t)nr * nr; ++i) Mc[i] = (double)acc[i];
    for (int i = 0; i < nr; ++i) rc[i] = (double)ar[i];
    free(map); free(wgt); free(acc); free(ar);
}

void orc_cpr_expand(int L, int basis, int DK, int DB, const double *cr, double *c) {
    int n = orc_num_unknowns(L, basis, DK, DB);
    int *map = (int *)malloc(sizeof(int) * n);
    double *wgt = (double *)malloc(sizeof(double) * n);
    cpr_map(L, basis, DK, DB, map, wgt);
    for (int k = 0; k < n; ++k) c[k] = wgt[k] * cr[map[k]];
    free(map); free(wgt);
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * NEXT-2: crowded-flavor preprocessing.  "The crowded-flavor SFFT will automatically mask the
 * pixels affected by the saturated sources in the field and replace them with the neighboring background."
 * The paper fixes neither the mask growth nor the background estimate; reading DESIGN g21:
 *   seed(x,y)  = R(x,y) >= sat_R  or  S(x,y) >= sat_S                 (one joint mask for the pair)
 *   mask(x,y)  = 1 iff some seed lies within Chebyshev distance rd     (square (2 rd + 1)^2 window)
 *   fill       : every masked pixel of an image <- mean of the UNMASKED pixels of that image inside the square
 *                (2 rb + 1)^2 window centred on it; if that window holds no unmasked pixel, the mean of all
 *                unmasked pixels of the image; unmasked pixels are copied.
 * Indices wrap around (the method is circular everywhere, DESIGN g12).  Plain loops, the definition itself.
 * Returns the number of masked pixels. */
long orc_mask_fill(int H, int W, const double *R, const double *S, double sat_R, double sat_S, int rd, int rb,
                   double *Rm, double *Sm, unsigned char *mask) {
    size_t P = (size_t)H * W;
    long nmask = 0;
    for (int x = 0; x < H; ++x)
        for (int y = 0; y < W; ++y) {
            int m = 0;
            for (int dx = -rd; dx <= rd && !m; ++dx)
                for (int dy = -rd; dy <= rd; ++dy) {
                    size_t q = (size_t)wrap(x + dx, H) * W + wrap(y + dy, W);
                    if (R[q] >= sat_R || S[q] >= sat_S) { m = 1; break; }
                }
            mask[(size_t)x * W + y] = (unsigned char)m;
            nmask += m;
        }
    const double *src[2] = {R, S};
    double *dst[2] = {Rm, Sm};
    for (int im = 0; im < 2; ++im) {
        long double gs = 0.0L; long gc = 0;
        for (size_t p = 0; p < P; ++p) if (!mask[p]) { gs += src[im][p]; ++gc; }
        double gmean = gc > 0 ? (double)(gs / gc) : 0.0;
#pragma omp parallel for schedule(dynamic, 8)
        for (int x = 0; x < H; ++x)
            for (int y = 0; y < W; ++y) {
                size_t p = (size_t)x * W + y;
                if (!mask[p]) { dst[im][p] = src[im][p]; continue; }
                long double s = 0.0L; long c = 0;
                for (int dx = -rb; dx <= rb; ++dx)
                    for (int dy = -rb; dy <= rb; ++dy) {
                        size_t q = (size_t)wrap(x + dx, H) * W + wrap(y + dy, W);
                        if (!mask[q]) { s += src[im][q]; ++c; }
                    }
                dst[im][p] = c > 0 ? (double)(s / c) : gmean;
            }
    }
    return nmask;
}
