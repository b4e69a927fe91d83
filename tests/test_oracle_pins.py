"""Pins for the CPU oracle (oracle/sfft_oracle.c) against things OTHER than itself:
the paper's Eqs. 14 and 19-24 evaluated literally with a library DFT, closed forms,
library routines (scipy.ndimage wrap-convolution, numpy lstsq, scipy BSpline), exact
rational arithmetic, and recovery of injected parameters.  CPU only.
Each test names the plausible mistake it would catch.
"""
import os
from fractions import Fraction

import numpy as np
import pytest
import scipy.interpolate
import scipy.ndimage

import oracle

POLY, BSPL = oracle.POLY, oracle.BSPLINE


def _u(N):
    return (2.0 * np.arange(N) + 1.0) / N - 1.0


def _poly_terms(D):
    return [(i, j) for i in range(D + 1) for j in range(D + 1 - i)]


def _poly_T(H, W, D):
    ux, uy = _u(H)[:, None], _u(W)[None, :]
    return [ux ** i * uy ** j * np.ones((H, W)) for (i, j) in _poly_terms(D)]


def _rand_pair(H, W, seed):
    rng = np.random.default_rng(seed)
    R = 100.0 + 50.0 * rng.random((H, W)) + 400.0 * (rng.random((H, W)) > 0.97)
    S = 90.0 + 60.0 * rng.random((H, W))
    return R, S


# --------------------------------------------------------------------------- weights

def test_term_order_and_counts():
    # i in [0,D], j in [0,D-i]  -> (D+1)(D+2)/2 terms; BASELINE unknown counts
    assert oracle.terms(POLY, 2) == [(0, 0), (0, 1), (0, 2), (1, 0), (1, 1), (2, 0)]
    golden = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "unknown_counts.txt")
    rows = [tuple(int(v) for v in ln.split()) for ln in open(golden) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 4
    for L, DK, DB, n in rows:
        assert oracle.num_unknowns(L, POLY, DK, DB) == n
        assert oracle.cpr_num_unknowns(L, POLY, DK, DB) == n - ((DK + 1) * (DK + 2) // 2 - 1)
    assert oracle.num_unknowns(11, BSPL, 4, 4) == 7808   # DESIGN g13: 8x8 functions
    assert oracle.terms(BSPL, 4)[9] == (1, 1)


def test_poly_axis_closed_form():
    for N in (8, 12, 128):
        tab = oracle.axis_table(POLY, N, 3)
        u = _u(N)
        for f in range(4):
            np.testing.assert_allclose(tab[f], u ** f, rtol=0, atol=2e-16)
        assert np.all(np.abs(u) < 1.0) and abs(u[0] + u[-1]) < 1e-15   # symmetric, inside (-1,1)


@pytest.mark.parametrize("N,m", [(16, 0), (64, 4), (100, 2), (1024, 4)])
def test_bspline_axis_vs_scipy(N, m):
    # catches a wrong knot vector, degree, or interval convention
    tab = oracle.axis_table(BSPL, N, m)
    knots = np.r_[np.zeros(4), np.arange(1, m + 1) / (m + 1.0), np.ones(4)]
    v = (np.arange(N) + 0.5) / N
    ref = scipy.interpolate.BSpline.design_matrix(v, knots, 3).toarray().T
    assert tab.shape == (m + 4, N)
    np.testing.assert_allclose(tab, ref, rtol=0, atol=5e-16)
    np.testing.assert_allclose(tab.sum(axis=0), 1.0, rtol=0, atol=1e-15)   # partition of unity
    assert tab.min() >= 0.0


# --------------------------------------------------------------------------- paper's equations

def test_eqs_14_19_24_literal_dft():
    """Evaluate Eqs. (14), (19)-(24) exactly as printed with numpy's FFT (forward DFT carrying
    1/(N0 N1), W = exp(-2 pi i/N)) and compare with the oracle's real-space normal system through
    A = M_aa/N^3, B = M_ab/N^2, C = M_bb/N, D = rhs_a/N^2, E = rhs_b/N  (N = N0 N1), and check that
    the paper's solution a = N * a_ring.  Catches: wrong shift sign, a dropped
    '-delta' term, transposed axes, wrong centre handling, wrong index order."""
    H, W, L, DK, DB = 12, 10, 3, 1, 1
    w, N = 1, H * W
    R, S = _rand_pair(H, W, 1)
    dft = lambda f: np.fft.fft2(f) / N
    l, m = np.arange(H)[:, None], np.arange(W)[None, :]
    W0, W1 = np.exp(-2j * np.pi / H), np.exp(-2j * np.pi / W)
    Khat = {}
    for al in range(-w, w + 1):
        for be in range(-w, w + 1):
            Khat[(al, be)] = np.full((H, W), 1.0 / N, complex) if (al, be) == (0, 0) \
                else (W0 ** (l * al) * W1 ** (m * be) - 1.0) / N
    TK, TB = _poly_T(H, W, DK), _poly_T(H, W, DB)
    Rhat = [dft(T * R) for T in TK]
    That = [dft(T) for T in TB]
    Shat = dft(S)
    lags = [(al, be) for al in range(-w, w + 1) for be in range(-w, w + 1)]
    FK, FB, LL = len(TK), len(TB), L * L
    n = FK * LL + FB
    Mp, rp = np.zeros((n, n)), np.zeros(n)
    for tb in range(FK):
        for ab, lb in enumerate(lags):
            kb = tb * LL + ab
            Xb = Rhat[tb] * Khat[lb]
            for t in range(FK):
                for a, la in enumerate(lags):
                    Mp[kb, t * LL + a] = np.sum((Xb * np.conj(Rhat[t]) * np.conj(Khat[la])).real)      # (19)
            for s in range(FB):
                Mp[kb, FK * LL + s] = np.sum((Xb * np.conj(That[s])).real)                              # (20)
                Mp[FK * LL + s, kb] = np.sum((That[s] * np.conj(Rhat[tb]) * np.conj(Khat[lb])).real)    # (21)
            rp[kb] = np.sum((np.conj(Shat) * Xb).real)                                                  # (23)
    for sb in range(FB):
        for s in range(FB):
            Mp[FK * LL + sb, FK * LL + s] = np.sum((That[sb] * np.conj(That[s])).real)                  # (22)
        rp[FK * LL + sb] = np.sum((np.conj(Shat) * That[sb]).real)                                      # (24)

    for M, rhs in (oracle.normal_bruteforce(R, S, L, POLY, DK, DB), oracle.normal_from_lags(R, S, L, POLY, DK, DB)):
        na = FK * LL
        sc = np.r_[np.full(na, float(N) ** 1.5), np.full(FB, float(N) ** 0.5)]
        Mo = M / np.outer(sc, sc)
        ro = rhs / np.r_[np.full(na, float(N) ** 2), np.full(FB, float(N))]
        scale = np.sqrt(np.outer(np.diag(Mp), np.diag(Mp)))
        assert np.max(np.abs(Mo - Mp) / scale) < 1e-13
        assert np.max(np.abs(ro - rp)) < 1e-13 * np.max(np.abs(rp))
        c = oracle.solve(M, rhs)
        cp = np.linalg.solve(Mp, rp)
        np.testing.assert_allclose(cp[:na] / N, c[:na], rtol=0, atol=1e-9 * np.abs(c).max())
        np.testing.assert_allclose(cp[na:], c[na:], rtol=0, atol=1e-9 * np.abs(c).max())


# --------------------------------------------------------------------------- structure of M

@pytest.mark.parametrize("H,W,L,basis,DK,DB", [(16, 12, 3, POLY, 1, 1), (12, 20, 5, POLY, 2, 1),
                                              (24, 16, 3, BSPL, 0, 0), (16, 16, 5, POLY, 0, 2)])
def test_tierB_equals_tierA_and_symmetric_psd(H, W, L, basis, DK, DB):
    R, S = _rand_pair(H, W, 2)
    MA, rA = oracle.normal_bruteforce(R, S, L, basis, DK, DB)
    MB, rB = oracle.normal_from_lags(R, S, L, basis, DK, DB)
    d = np.sqrt(np.diag(MA))
    assert np.max(np.abs(MA - MB) / np.outer(d, d)) < 1e-13
    assert np.max(np.abs(rA - rB)) < 1e-13 * np.max(np.abs(rA))
    assert np.array_equal(MA, MA.T) and np.array_equal(MB, MB.T)
    assert np.linalg.eigvalsh(MA / np.outer(d, d)).min() > -1e-12


def test_tierA_vs_independent_numpy_design_matrix():
    """Phi rebuilt with np.roll from Eqs. 3-4, 11 (independent of the C loops), M = Phi^T Phi via BLAS."""
    H, W, L, DK, DB = 16, 20, 5, 2, 1
    w = 2
    R, S = _rand_pair(H, W, 3)
    cols = []
    for T in _poly_T(H, W, DK):
        Rt = T * R
        for al in range(-w, w + 1):
            for be in range(-w, w + 1):
                sh = np.roll(Rt, (al, be), axis=(0, 1))          # sh(x,y) = Rt(x-al, y-be)
                cols.append((sh if (al, be) == (0, 0) else sh - Rt).ravel())
    cols += [T.ravel() for T in _poly_T(H, W, DB)]
    Phi = np.array(cols)
    np.testing.assert_allclose(oracle.design_matrix(R, L, POLY, DK, DB), Phi, rtol=0, atol=1e-12)
    M, rhs = oracle.normal_bruteforce(R, S, L, POLY, DK, DB)
    np.testing.assert_allclose(M, Phi @ Phi.T, rtol=1e-12, atol=1e-6)
    np.testing.assert_allclose(rhs, Phi @ S.ravel(), rtol=1e-12, atol=1e-6)


def test_background_block_exact_rational():
    """M_bb = products of power sums of the normalised coordinates, in exact Fractions;
    rhs_b = image moments of S.  Catches wrong coordinates or term order in the background block."""
    H, W, L, DB = 12, 8, 3, 2
    R, S = _rand_pair(H, W, 4)
    M, rhs = oracle.normal_from_lags(R, S, L, POLY, 0, DB)
    ps = lambda N, k: sum((Fraction(2 * x + 1, N) - 1) ** k for x in range(N))
    tb = _poly_terms(DB)
    for a, (ib, jb) in enumerate(tb):
        for b, (i, j) in enumerate(tb):
            exact = float(ps(H, ib + i) * ps(W, jb + j))
            assert abs(M[L * L + a, L * L + b] - exact) <= 1e-14 * max(1.0, abs(exact))
        mom = np.sum(S * _u(H)[:, None] ** ib * _u(W)[None, :] ** jb)
        assert abs(rhs[L * L + a] - mom) <= 1e-12 * np.abs(S).sum()


def test_lag_symmetries():
    H, W, L = 16, 12, 3
    R, S = _rand_pair(H, W, 5)
    t = oracle.lag_tables(R, S, L, POLY, 1, 1)
    A, B = oracle.weighted_ref(R, POLY, 1, 0), oracle.weighted_ref(R, POLY, 1, 2)
    for rho, eps in [(1, -2), (-2, 0), (0, 1), (2, 2)]:
        q, c0 = oracle.corr_diff_one(A, B, rho, eps)
        qr, c0r = oracle.corr_diff_one(B, A, -rho, -eps)
        assert abs((q + c0) - (qr + c0r)) < 1e-9 * abs(c0)                       # Omega_ab(r) = Omega_ba(-r)
        assert abs(q - t["Qom"][0, 2, rho + 2, eps + 2]) < 1e-9 * abs(c0)
        direct = np.sum(A * np.roll(B, (-rho, -eps), axis=(0, 1)))                 # B(x+rho, y+eps)
        assert abs((q + c0) - direct) < 1e-12 * abs(direct)
    q00 = t["Qom"][0, 0]
    np.testing.assert_allclose(q00, q00[::-1, ::-1], rtol=0, atol=1e-9 * t["Om0"][0, 0])   # Omega_tt even


# --------------------------------------------------------------------------- solution

def test_solve_vs_lapack_and_not_spd():
    rng = np.random.default_rng(6)
    X = rng.standard_normal((200, 40)) * np.logspace(0, 4, 40)[None, :]
    M, c_true = X.T @ X, rng.standard_normal(40)
    c = oracle.solve(M, M @ c_true)
    np.testing.assert_allclose(c, np.linalg.solve(M, M @ c_true), rtol=1e-9, atol=1e-12)
    np.testing.assert_allclose(c, c_true, rtol=1e-9, atol=1e-12)
    M[5, 5] = -1.0
    with pytest.raises(np.linalg.LinAlgError):
        oracle.solve(M, M @ c_true)


def test_solution_vs_lstsq_qr():
    """c from the oracle's normal equations == QR/SVD least squares on Phi (never forms M)."""
    H, W, L, DK, DB = 20, 16, 3, 1, 1
    R, S = _rand_pair(H, W, 7)
    Phi = oracle.design_matrix(R, L, POLY, DK, DB)
    c_ls = np.linalg.lstsq(Phi.T, S.ravel(), rcond=None)[0]
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, POLY, DK, DB))
    np.testing.assert_allclose(c, c_ls, rtol=0, atol=1e-10 * np.abs(c_ls).max())


def test_identical_images_give_delta_kernel_and_zero_difference():
    H, W, L = 16, 16, 5
    R, _ = _rand_pair(H, W, 8)
    c = oracle.solve(*oracle.normal_from_lags(R, R, L, POLY, 1, 1))
    e = np.zeros_like(c); e[(L // 2) * L + L // 2] = 1.0
    np.testing.assert_allclose(c, e, rtol=0, atol=1e-10)
    assert np.abs(oracle.difference(R, R, c, L, POLY, 1, 1)).max() < 1e-9


def test_shift_scale_constant_recovered():
    """S = lam * R(x-1, y+1) + mu  =>  a_{0,centre} = lam (kernel sum), a_{0,(1,-1)} = lam, b_0 = mu, rest 0."""
    H, W, L, lam, mu = 16, 20, 3, 1.1, 3.0
    R, _ = _rand_pair(H, W, 9)
    S = lam * np.roll(R, (1, -1), axis=(0, 1)) + mu
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, POLY, 1, 1))
    expect = np.zeros_like(c)
    expect[1 * L + 1] = lam                    # centre
    expect[(1 + 1) * L + (-1 + 1)] = lam       # (alpha,beta) = (1,-1)
    expect[3 * L * L] = mu
    np.testing.assert_allclose(c, expect, rtol=0, atol=1e-9)


def test_constant_kernel_is_textbook_circular_convolution():
    """App. A: for DK=0 the model is an exact circular convolution.  S is made by
    scipy.ndimage.convolve(mode='wrap'); the oracle must return that kernel, and its difference
    routine must reproduce scipy's convolution."""
    H, W, L = 24, 20, 5
    rng = np.random.default_rng(10)
    R, _ = _rand_pair(H, W, 10)
    k = rng.random((L, L)); k[0, 3] = 0.9            # asymmetric on purpose
    S = scipy.ndimage.convolve(R, k, mode="wrap") + 7.0
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, POLY, 0, 0))
    kc = c[:L * L].reshape(L, L).copy()
    ksum = kc[2, 2]
    kc[2, 2] = ksum - (kc.sum() - ksum)              # Eqs. 3-4: centre coefficient is the kernel SUM
    np.testing.assert_allclose(kc, k, rtol=0, atol=1e-9)
    assert abs(ksum - k.sum()) < 1e-9 and abs(c[-1] - 7.0) < 1e-8
    D = oracle.difference(R, np.zeros_like(R), c, L, POLY, 0, 0)
    np.testing.assert_allclose(-D, S, rtol=0, atol=1e-9)


@pytest.mark.parametrize("basis,DK,DB", [(POLY, 2, 1), (BSPL, 0, 0)])
def test_injected_spatially_varying_model_recovered(basis, DK, DB):
    """S = sum_t (T_t R) o k_t + sum_s b_s T'_s  built with scipy's wrap-convolution per term
    (Eq. 12) from chosen kernels; the fit must return them (noiseless => exact)."""
    H, W, L = 32, 28, 3
    rng = np.random.default_rng(11)
    R, _ = _rand_pair(H, W, 11)
    if basis == POLY:
        TK, TB = _poly_T(H, W, DK), _poly_T(H, W, DB)
    else:
        fx, gy = oracle.axis_table(BSPL, H, DK), oracle.axis_table(BSPL, W, DK)   # pinned to scipy above
        TK = [np.outer(fx[i], gy[j]) for (i, j) in oracle.terms(BSPL, DK)]
        TB = TK
    ks = [rng.standard_normal((L, L)) * (1.0 if t == 0 else 0.2) for t in range(len(TK))]
    bs = rng.standard_normal(len(TB))
    S = sum(scipy.ndimage.convolve(T * R, k, mode="wrap") for T, k in zip(TK, ks)) + sum(b * T for b, T in zip(bs, TB))
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, basis, DK, DB))
    LL = L * L
    for t, k in enumerate(ks):
        a = k.ravel().copy(); a[LL // 2] = k.sum()
        np.testing.assert_allclose(c[t * LL:(t + 1) * LL], a, rtol=0, atol=2e-8)
    np.testing.assert_allclose(c[len(TK) * LL:], bs, rtol=0, atol=1e-6)
    D = oracle.difference(R, S, c, L, basis, DK, DB)
    assert np.abs(D).max() < 1e-7


def test_kernel_sum_property_with_delta_image():
    """the kernel sum at a position is the K_00 coefficient field sum_t a_{t,00} T_t.
    A delta image at (x0,y0) makes the model image equal the local kernel (weights at the source pixel)."""
    H, W, L, DK = 16, 16, 3, 1
    rng = np.random.default_rng(12)
    n = oracle.num_unknowns(L, POLY, DK, 0)
    c = rng.standard_normal(n); c[-1] = 0.0
    x0, y0 = 5, 9
    R = np.zeros((H, W)); R[x0, y0] = 1.0
    model = -oracle.difference(R, np.zeros((H, W)), c, L, POLY, DK, 0)
    T = [Tt[x0, y0] for Tt in _poly_T(H, W, DK)]
    expect_sum = sum(c[t * L * L + L * L // 2] * T[t] for t in range(3))
    assert abs(model.sum() - expect_sum) < 1e-12
    a_off = sum(c[t * L * L + (1 + 1) * L + (0 + 1)] * T[t] for t in range(3))   # (alpha,beta) = (1,0)
    assert abs(model[x0 + 1, y0] - a_off) < 1e-12


def test_normal_equation_orthogonality_and_sampled_difference():
    H, W, L = 20, 24, 5
    R, S = _rand_pair(H, W, 13)
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, POLY, 1, 1))
    D = oracle.difference(R, S, c, L, POLY, 1, 1)
    Phi = oracle.design_matrix(R, L, POLY, 1, 1)
    g = Phi @ D.ravel()
    assert np.max(np.abs(g) / (np.linalg.norm(Phi, axis=1) * np.linalg.norm(D))) < 1e-11
    px, py = np.array([0, 3, 19, 7]), np.array([0, 23, 11, 2])
    np.testing.assert_allclose(oracle.difference_at(R, S, c, L, POLY, 1, 1, px, py), D[px, py], rtol=0, atol=1e-10)


def _numpy_design(R, L, basis, DK, DB):
    """Design matrix rebuilt with np.roll (Eqs. 3-4, 11), weights from closed forms (POLY) or scipy (BSPLINE)."""
    H, W = R.shape
    w = (L - 1) // 2
    if basis == POLY:
        TK, TB = _poly_T(H, W, DK), _poly_T(H, W, DB)
    else:
        def ax(N, m):
            knots = np.r_[np.zeros(4), np.arange(1, m + 1) / (m + 1.0), np.ones(4)]
            return scipy.interpolate.BSpline.design_matrix((np.arange(N) + 0.5) / N, knots, 3).toarray().T
        fK, gK, fB, gB = ax(H, DK), ax(W, DK), ax(H, DB), ax(W, DB)
        TK = [np.outer(fK[i], gK[j]) for i in range(DK + 4) for j in range(DK + 4)]
        TB = [np.outer(fB[i], gB[j]) for i in range(DB + 4) for j in range(DB + 4)]
    cols = []
    for T in TK:
        Rt = T * R
        for al in range(-w, w + 1):
            for be in range(-w, w + 1):
                sh = np.roll(Rt, (al, be), axis=(0, 1))
                cols.append((sh if (al, be) == (0, 0) else sh - Rt).ravel())
    cols += [T.ravel() for T in TB]
    return np.array(cols)


@pytest.mark.parametrize("H,W,L,basis,DK,DB", [(20, 24, 5, POLY, 2, 1), (24, 20, 5, BSPL, 1, 0), (16, 16, 7, BSPL, 0, 1)])
def test_difference_at_on_borders_and_diag_rhs_vs_numpy(H, W, L, basis, DK, DB):
    """orc_difference_at (the sampled form the full-size configs rest on) against D = S - Phi^T c with Phi rebuilt
    in numpy, at pixels whose kernel footprint wraps in x, in y and in both (all four corners), under both bases;
    catches a wrong wrap direction, a transposed weight table or a missing centre correction.
    orc_diag_and_rhs against the same Phi (catches a wrong shift sign or a dropped '- R^t' term)."""
    R, S = _rand_pair(H, W, 21)
    Phi = _numpy_design(R, L, basis, DK, DB)
    rng = np.random.default_rng(22)
    c = rng.standard_normal(Phi.shape[0])
    D = (S.ravel() - c @ Phi).reshape(H, W)
    px = np.array([0, 0, H - 1, H - 1, 1, H - 2, H // 2, 0, H - 1, 3])
    py = np.array([0, W - 1, 0, W - 1, W - 2, 1, W // 2, W // 2, 2, 0])
    np.testing.assert_allclose(oracle.difference_at(R, S, c, L, basis, DK, DB, px, py), D[px, py], rtol=0, atol=2e-10)
    np.testing.assert_allclose(oracle.difference(R, S, c, L, basis, DK, DB), D, rtol=0, atol=2e-10)
    diag, rhs = oracle.diag_and_rhs(R, S, L, basis, DK, DB)
    np.testing.assert_allclose(diag, np.sum(Phi * Phi, axis=1), rtol=1e-12, atol=1e-9)
    np.testing.assert_allclose(rhs, Phi @ S.ravel(), rtol=1e-12, atol=1e-7)


def test_affine_coordinate_invariance_of_difference():
    """DESIGN g8: the total-degree polynomial space is affine invariant, so D fitted with raw pixel
    indices (the paper's T = x^p y^q) equals D fitted with normalised coordinates."""
    H, W, L, DK, DB = 16, 12, 3, 1, 1
    R, S = _rand_pair(H, W, 14)
    c = oracle.solve(*oracle.normal_from_lags(R, S, L, POLY, DK, DB))
    D = oracle.difference(R, S, c, L, POLY, DK, DB)
    x, y = np.arange(H)[:, None] * 1.0, np.arange(W)[None, :] * 1.0
    raw = [x ** i * y ** j * np.ones((H, W)) for (i, j) in _poly_terms(1)]
    cols = []
    for T in raw:
        Rt = T * R
        for al in (-1, 0, 1):
            for be in (-1, 0, 1):
                sh = np.roll(Rt, (al, be), axis=(0, 1))
                cols.append((sh if (al, be) == (0, 0) else sh - Rt).ravel())
    cols += [T.ravel() for T in raw]
    Phi = np.array(cols).T
    c_raw = np.linalg.lstsq(Phi, S.ravel(), rcond=None)[0]
    np.testing.assert_allclose(D.ravel(), S.ravel() - Phi @ c_raw, rtol=0, atol=1e-8)


# --------------------------------------------------------------------------- NEXT-1: constant photometric ratio

def _cpr_design(R, L, basis, DK, DB):
    """Design matrix of the constant-kernel-integral model written from PAPER.md:121 directly: the F_K centre
    columns R^t are replaced by ONE column, the unweighted reference R (the kernel integral multiplies R itself)."""
    Phi = oracle.design_matrix(R, L, basis, DK, DB)
    FK, LL, a0 = oracle.num_terms(basis, DK), L * L, (L // 2) * L + L // 2
    keep = [k for k in range(Phi.shape[0]) if not (k < FK * LL and k % LL == a0 and k >= LL)]
    Phir = Phi[keep].copy()
    Phir[a0] = R.ravel()
    return Phir


@pytest.mark.parametrize("basis,DK,DB", [(POLY, 1, 1), (POLY, 2, 0), (BSPL, 1, 0)])
def test_cpr_system_and_solution_vs_bruteforce_lstsq(basis, DK, DB):
    """Catches a wrong index map (which centre entries merge), a wrong weight (zero vs one) and a transposed C."""
    H, W, L = 14, 18, 3
    R, S = _rand_pair(H, W, 21)
    M, rhs = oracle.normal_from_lags(R, S, L, basis, DK, DB)
    Mc, rc = oracle.cpr_constrain(M, rhs, L, basis, DK, DB)
    Phir = _cpr_design(R, L, basis, DK, DB)
    assert Mc.shape[0] == Phir.shape[0] == oracle.cpr_num_unknowns(L, basis, DK, DB)
    assert np.allclose(Mc, Phir @ Phir.T, rtol=1e-11, atol=1e-8 * np.abs(Mc).max() * 1e-3)
    assert np.allclose(rc, Phir @ S.ravel(), rtol=1e-11)
    cr = oracle.solve(Mc, rc)
    ref = np.linalg.lstsq(Phir.T, S.ravel(), rcond=None)[0]
    assert np.max(np.abs(cr - ref)) <= 1e-8 * np.max(np.abs(ref))
    # expansion reproduces the same model image
    c = oracle.cpr_expand(cr, L, basis, DK, DB)
    Phi = oracle.design_matrix(R, L, basis, DK, DB)
    assert np.allclose(Phi.T @ c, Phir.T @ cr, rtol=1e-12, atol=1e-9)


@pytest.mark.parametrize("basis,DK", [(POLY, 2), (BSPL, 1)])
def test_cpr_kernel_integral_is_constant_over_the_field(basis, DK):
    """A_xy00 = a_0000.  The kernel-sum field sum_t a_{t,00} T_t(x,y) of the expanded solution must
    not depend on (x, y) and must equal the shared unknown."""
    H, W, L, DB = 16, 16, 3, 1
    R, S = _rand_pair(H, W, 22)
    M, rhs = oracle.normal_from_lags(R, S, L, basis, DK, DB)
    cr = oracle.solve(*oracle.cpr_constrain(M, rhs, L, basis, DK, DB))
    c = oracle.cpr_expand(cr, L, basis, DK, DB)
    fx, gy = oracle.axis_table(basis, H, DK), oracle.axis_table(basis, W, DK)
    a0, LL = (L // 2) * L + L // 2, L * L
    field = sum(c[t * LL + a0] * np.outer(fx[i], gy[j]) for t, (i, j) in enumerate(oracle.terms(basis, DK)))
    assert np.allclose(field, cr[a0], rtol=1e-12, atol=1e-12)


def test_cpr_recovers_constant_scale_with_varying_kernel():
    """Noiseless S = 1.25 * (R convolved with a kernel whose SHAPE varies linearly in x but whose sum is 1) + 7:
    the constrained fit recovers the scale 1.25 as the shared unknown and leaves a zero difference."""
    H, W, L, DK, DB = 24, 24, 3, 1, 0
    rng = np.random.default_rng(5)
    R = 100.0 + 50.0 * rng.random((H, W))
    ux = _u(H)[:, None] * np.ones((1, W))
    # model image built from the definition: scale * [R + g(x) * (shifted copies - R)], g = 0.2 + 0.1 u_x at the source pixel
    g = 0.2 + 0.1 * ux
    Rg = R * g
    S = 1.25 * (R + (np.roll(Rg, (1, 0), (0, 1)) - Rg) + (np.roll(Rg, (0, -1), (0, 1)) - Rg)) + 7.0
    M, rhs = oracle.normal_from_lags(R, S, L, POLY, DK, DB)
    cr = oracle.solve(*oracle.cpr_constrain(M, rhs, L, POLY, DK, DB))
    a0 = (L // 2) * L + L // 2
    assert abs(cr[a0] - 1.25) <= 1e-9
    c = oracle.cpr_expand(cr, L, POLY, DK, DB)
    assert np.max(np.abs(oracle.difference(R, S, c, L, POLY, DK, DB))) <= 1e-8


# --------------------------------------------------------------------------- NEXT-2: crowded-flavor mask + fill

def _saturated_pair(H, W, seed, sat=600.0):
    rng = np.random.default_rng(seed)
    R = 100.0 + 20.0 * rng.random((H, W))
    S = 110.0 + 20.0 * rng.random((H, W))
    for (x, y, a) in [(5, 7, 900.0), (H - 1, 0, 1500.0), (H // 2, W - 1, 700.0)]:      # two of them wrap around the frame
        R[x, y] = a
    S[3, W // 2] = 2000.0
    S[5, 7] = 650.0
    return R, S, sat


def test_mask_fill_golden_9x9():
    """Hand-computed example (tests/golden/mask_fill_9x9.txt, DESIGN g21): catches a wrong window size,
    masked pixels leaking into the mean, or a transposed axis."""
    x, y = np.meshgrid(np.arange(9.0), np.arange(9.0), indexing="ij")
    I = x + 10.0 * y
    I[4, 4] = 1000.0
    Rm, Sm, mask = oracle.mask_fill(I, np.zeros_like(I), 500.0, 500.0, 1, 2)
    expect = np.zeros((9, 9), np.uint8); expect[3:6, 3:6] = 1
    assert np.array_equal(mask, expect)
    golden = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "mask_fill_9x9.txt")
    rows = [ln.split() for ln in open(golden) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 5
    for gx, gy, val in rows:
        assert abs(Rm[int(gx), int(gy)] - float(val)) < 1e-12
    assert np.array_equal(Rm[mask == 0], I[mask == 0]) and np.array_equal(Sm[mask == 0], 0 * I[mask == 0])


@pytest.mark.parametrize("rd,rb", [(0, 1), (1, 3), (2, 5)])
def test_mask_fill_vs_scipy_filters_and_invariants(rd, rb):
    """mask = wrap-around maximum filter of the thresholded seed (library routine); fill = ratio of two wrap-around
    box filters (library routine); mask contains the thresholded set; filled values lie inside the range of the
    unmasked neighbourhood; an unsaturated pair comes back untouched (idempotence)."""
    H, W = 24, 20
    R, S, sat = _saturated_pair(H, W, 31)
    Rm, Sm, mask = oracle.mask_fill(R, S, sat, sat, rd, rb)
    seed = ((R >= sat) | (S >= sat)).astype(np.uint8)
    ref_mask = scipy.ndimage.maximum_filter(seed, size=2 * rd + 1, mode="wrap")
    assert np.array_equal(mask, ref_mask) and np.all(mask[seed == 1] == 1)
    keep = 1.0 - mask
    for I, Im in ((R, Rm), (S, Sm)):
        num = scipy.ndimage.uniform_filter(I * keep, size=2 * rb + 1, mode="wrap")
        den = scipy.ndimage.uniform_filter(keep, size=2 * rb + 1, mode="wrap")
        assert den[mask == 1].min() > 0
        np.testing.assert_allclose(Im[mask == 1], (num / den)[mask == 1], rtol=1e-12)
        assert np.array_equal(Im[mask == 0], I[mask == 0])
        lo = scipy.ndimage.minimum_filter(np.where(mask == 1, np.inf, I), size=2 * rb + 1, mode="wrap")
        hi = scipy.ndimage.maximum_filter(np.where(mask == 1, -np.inf, I), size=2 * rb + 1, mode="wrap")
        assert np.all(Im[mask == 1] >= lo[mask == 1] - 1e-12) and np.all(Im[mask == 1] <= hi[mask == 1] + 1e-12)
    R2, S2, m2 = oracle.mask_fill(Rm, Sm, sat, sat, rd, rb)          # nothing saturated any more
    assert m2.sum() == 0 and np.array_equal(R2, Rm) and np.array_equal(S2, Sm)


def test_mask_fill_empty_window_falls_back_to_global_mean():
    """A saturated blob larger than the fill window: pixels whose window holds no unmasked pixel take the mean of all
    unmasked pixels of the image."""
    H = W = 16
    R = 50.0 + np.arange(H * W, dtype=np.float64).reshape(H, W) % 7
    S = R + 1.0
    R[4:12, 4:12] = 1e4
    Rm, Sm, mask = oracle.mask_fill(R, S, 1e3, 1e3, 0, 1)
    assert mask.sum() == 64
    np.testing.assert_allclose(Rm[7, 7], R[mask == 0].mean(), rtol=1e-13)
    np.testing.assert_allclose(Sm[8, 8], S[mask == 0].mean(), rtol=1e-13)


# --------------------------------------------------------------------------- NEXT-3: noise decorrelation (App. C)

def _gauss_kernel(L, sig, shift=(0.0, 0.0)):
    w = (L - 1) // 2
    a = np.arange(-w, w + 1)
    k = np.exp(-0.5 * ((a[:, None] - shift[0]) ** 2 + (a[None, :] - shift[1]) ** 2) / sig ** 2)
    return k / k.sum()


def _coef_from_pixel_kernels(ks, FB=1):
    """Delta-basis coefficients whose pixel kernels (Eqs. 3-4) are ks[t]: centre coefficient = kernel sum."""
    out = []
    for k in ks:
        a = k.ravel().copy()
        a[a.size // 2] = k.sum()
        out.append(a)
    return np.concatenate(out + [np.zeros(FB)])


def test_decorrelation_delta_kernel_is_identity_and_c20_values():
    """K = c * delta, G = H = delta  =>  the C20 denominator is flat, Q0^ = 1, the image comes back unchanged.
    And C20 itself at a few frequencies with K^ summed straight from its definition (no FFT): catches a wrong
    sign/normalisation of the kernel transform, a missing square, or swapped variances."""
    from oracle import decorr
    rng = np.random.default_rng(41)
    D = rng.standard_normal((64, 64))
    L = 5
    kd = np.zeros((L, L)); kd[2, 2] = 1.7
    coef = _coef_from_pixel_kernels([kd])
    out = decorr.decorrelate(D, coef, L, POLY, 0, 32, [2.0], [[[1.0]]], [3.0], [[[1.0]]])
    np.testing.assert_allclose(out, D, rtol=0, atol=1e-13)
    K = _gauss_kernel(L, 1.1, (0.3, -0.2)) * 0.9
    Hk = _gauss_kernel(3, 0.8) / 2.0
    T = 16
    Q0, den = decorr.q0_hat(K, T, [2.0, 1.5], [[[0.5]], [[0.5]]], [3.0, 2.5], [Hk, Hk])
    a = np.arange(-2, 3)
    for (l, m) in [(0, 0), (1, 0), (3, 5), (8, 8), (15, 2)]:
        Kh = np.sum(K * np.exp(-2j * np.pi * (l * a[:, None] + m * a[None, :]) / T))
        ah = np.arange(-1, 2)
        Hh = np.sum(Hk * np.exp(-2j * np.pi * (l * ah[:, None] + m * ah[None, :]) / T))
        d = (2.0 + 1.5) * 0.25 + abs(Kh) ** 2 * (3.0 + 2.5) * abs(Hh) ** 2
        assert abs(den[l, m] - d) < 1e-13 * d
    d0 = (2.0 + 1.5) * 0.25 + K.sum() ** 2 * (3.0 + 2.5) * Hk.sum() ** 2
    assert abs(Q0[3, 5] - np.sqrt(d0 / den[3, 5])) < 1e-14 and abs(Q0[0, 0] - 1.0) < 1e-15


def test_decorrelation_kernel_has_unit_sum_and_is_a_wrap_convolution():
    """Q has unit sum.  The response to a delta image IS Q; convolving with that Q through an
    independent routine (scipy wrap convolution) must reproduce the tile-wise output: checks linearity, shift
    invariance inside a tile, tile independence and the frozen-at-tile-centre kernel (spatially varying fit)."""
    from oracle import decorr
    H = W = 64; T = 32; L = 5
    k0, k1 = _gauss_kernel(L, 1.0), _gauss_kernel(L, 1.6, (0.4, 0.0)) - _gauss_kernel(L, 1.0)
    coef = np.concatenate([_coef_from_pixel_kernels([k0, 0.3 * k1, -0.2 * k1], FB=0), np.zeros(3)])   # DK = 1: 3 terms
    args = (coef, L, POLY, 1, T, [1.0], [[[1.0]]], [1.3], [[[1.0]]])
    rng = np.random.default_rng(42)
    D = rng.standard_normal((H, W))
    out = decorr.decorrelate(D, *args)
    for a in range(2):
        for b in range(2):
            imp = np.zeros((H, W)); imp[a * T + T // 2, b * T + T // 2] = 1.0
            Q = decorr.decorrelate(imp, *args)[a * T:(a + 1) * T, b * T:(b + 1) * T]     # centred at (T/2, T/2)
            assert abs(Q.sum() - 1.0) < 1e-13
            np.testing.assert_allclose(Q[1:, 1:], Q[1:, 1:][::-1, ::-1], atol=1e-14)    # Q(-u) = Q(u): Q0^ is real
            ref = scipy.ndimage.convolve(D[a * T:(a + 1) * T, b * T:(b + 1) * T], Q, mode="wrap", origin=0)
            np.testing.assert_allclose(out[a * T:(a + 1) * T, b * T:(b + 1) * T], ref, rtol=0, atol=1e-12)
    # the kernel differs between tiles (spatial variation of the fit)
    assert np.abs(decorr.kernel_at(coef, L, POLY, 1, H, W, 16, 16) - decorr.kernel_at(coef, L, POLY, 1, H, W, 48, 48)).max() > 1e-3
    # kernel_at against the model of the difference image: -D of a delta reference at (xc,yc) read around (xc,yc)
    R = np.zeros((H, W)); R[16, 16] = 1.0
    model = -oracle.difference(R, np.zeros((H, W)), coef, L, POLY, 1, 1)
    np.testing.assert_allclose(model[14:19, 14:19], decorr.kernel_at(coef, L, POLY, 1, H, W, 16, 16), atol=1e-14)


def test_decorrelation_whitens_the_noise():
    """Statistical pin (App. C's purpose): D = n_S - n_R (*) K with white n_S, n_R has correlated noise; after
    decorrelation the sample autocorrelation at small lags vanishes to sampling error and the variance is the
    C20 denominator at zero frequency, sigma_S^2 + sigma_R^2 (sum K)^2."""
    from oracle import decorr
    T = 128; L = 7
    rng = np.random.default_rng(43)
    K = _gauss_kernel(L, 1.4) * 1.1
    vS, vR = 4.0, 9.0
    nS, nR = rng.normal(0, np.sqrt(vS), (T, T)), rng.normal(0, np.sqrt(vR), (T, T))
    D = nS - scipy.ndimage.convolve(nR, K, mode="wrap")
    coef = _coef_from_pixel_kernels([K])
    out = decorr.decorrelate(D, coef, L, POLY, 0, T, [vS], [[[1.0]]], [vR], [[[1.0]]])

    def acorr(img, dx, dy):
        z = img - img.mean()
        return float(np.mean(z * np.roll(z, (dx, dy), axis=(0, 1))) / np.mean(z * z))
    assert abs(acorr(D, 0, 1)) > 0.05 and abs(acorr(D, 1, 1)) > 0.03           # correlated before (sampling error 1/T = 0.008)
    for lag in [(0, 1), (1, 0), (1, 1), (2, 0), (0, 3)]:
        assert abs(acorr(out, *lag)) < 5.0 / T                                     # white after (sampling error 1/T)
    assert abs(out.var() / (vS + vR * K.sum() ** 2) - 1.0) < 0.05


# --------------------------------------------------------------------------- NEXT-4: rectangular kernels

@pytest.mark.parametrize("L0,L1", [(3, 7), (5, 1)])
def test_rectangular_kernel_selection_vs_direct_design_matrix(L0, L1):
    """PAPER.md:86 (the delta basis spans L0 x L1 pixels): the oracle's rectangular system (a selection from the
    enclosing square's) against a design matrix built directly for the L0 x L1 lag set with np.roll, its Gram matrix
    and numpy lstsq; the expanded solution subtracts like the direct model.  Catches swapped axes (alpha <-> beta),
    a selection that keeps the wrong rows, and a wrong expansion."""
    H, W, DK, DB = 16, 20, 1, 1
    w0, w1 = (L0 - 1) // 2, (L1 - 1) // 2
    R, S = _rand_pair(H, W, 11)
    cols = []
    for T in _poly_T(H, W, DK):
        Rt = T * R
        for al in range(-w0, w0 + 1):
            for be in range(-w1, w1 + 1):
                sh = np.roll(Rt, (al, be), axis=(0, 1))          # sh(x,y) = Rt(x-al, y-be)
                cols.append((sh if (al, be) == (0, 0) else sh - Rt).ravel())
    cols += [T.ravel() for T in _poly_T(H, W, DB)]
    Phi = np.array(cols)
    L = max(L0, L1)
    sel = oracle.rect_select(L0, L1, POLY, DK, DB)
    assert len(sel) == Phi.shape[0] == 3 * L0 * L1 + 3 and np.all(np.diff(sel) > 0)
    M, rhs = oracle.normal_from_lags(R, S, L, POLY, DK, DB)
    Ms, rs = M[np.ix_(sel, sel)], rhs[sel]
    np.testing.assert_allclose(Ms, Phi @ Phi.T, rtol=1e-11, atol=1e-5)
    np.testing.assert_allclose(rs, Phi @ S.ravel(), rtol=1e-11, atol=1e-5)
    cs = oracle.solve(Ms, rs)
    cl = np.linalg.lstsq(Phi.T, S.ravel(), rcond=None)[0]
    np.testing.assert_allclose(cs, cl, rtol=0, atol=1e-9 * np.max(np.abs(cl)))
    D = oracle.difference(R, S, oracle.rect_expand(cs, L0, L1, POLY, DK, DB), L, POLY, DK, DB)
    np.testing.assert_allclose(D, S - (Phi.T @ cl).reshape(H, W), rtol=0, atol=1e-8)
