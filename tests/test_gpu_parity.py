"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's, in the DESIGN g16 reading:
  matrix   |dM_kk'| <= 1e-10 sqrt(M_kk M_k'k')      rhs |d rhs_k| <= 1e-10 sqrt(M_kk sum S^2)
  solution max|dc| <= 1e-8 max|c| per block (kernel, background)
  D        max|dD| <= 1e-6 sigma,  sigma = sqrt(sky + read^2) = sqrt(125) ADU
"""
import numpy as np
import pytest

import oracle
from paper_2109_09334_b200 import binding as B
import synth

pytestmark = pytest.mark.gpu

TOL_M, TOL_C, TOL_D = 1e-10, 1e-8, 1e-6


def _bid(basis):
    return oracle.POLY if basis == "poly" else oracle.BSPLINE


def _oracle_all(R, S, L, basis, DK, DB):
    bid = _bid(basis)
    M, rhs = oracle.normal_from_lags(R, S, L, bid, DK, DB)
    c = oracle.solve(M, rhs)
    D = oracle.difference(R, S, c, L, bid, DK, DB)
    return M, rhs, c, D


def _check_system(M, rhs, Mo, ro, S):
    d = np.sqrt(np.diag(Mo))
    assert np.max(np.abs(M - Mo) / np.outer(d, d)) <= TOL_M
    assert np.max(np.abs(rhs - ro) / (d * np.sqrt(np.sum(S * S)))) <= TOL_M
    assert np.array_equal(M, M.T)


def _check_coef(c, co, na):
    assert np.max(np.abs(c[:na] - co[:na])) <= TOL_C * np.max(np.abs(co[:na]))
    assert np.max(np.abs(c[na:] - co[na:])) <= TOL_C * np.max(np.abs(co[na:]))


def _gpu_all(torch, p, L, basis, DK, DB, R=None, S=None, corr_route=0, reuse_spectra=False):
    R = p.R if R is None else R
    S = p.S if S is None else S
    nb = 1 if R.ndim == 2 else R.shape[0]
    H, W = R.shape[-2:]
    plan = B.Plan(H, W, L, DK, DB, basis, nbatch=nb, corr_route=corr_route, reuse_spectra=reuse_spectra)
    dR, dS = torch.from_numpy(np.ascontiguousarray(R)).cuda(), torch.from_numpy(np.ascontiguousarray(S)).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    plan.status()
    M, rhs = plan.system()
    out = M.cpu().numpy(), rhs.cpu().numpy(), coef.cpu().numpy(), D.cpu().numpy()
    plan.close()
    return out


CASES = [
    # (config, H, W, L, basis, DK, DB)  -- None = the config's own value
    (1, None, None, None, None, None, None),          # config 1 as specified
    (2, 256, 256, None, None, None, None),            # config-2 recipe, several row tiles, L=11
    (2, 128, 512, 5, None, None, None),               # non-square
    (3, 64, 256, 15, None, None, None),               # 2L-1 = 29 lags on a small frame (wrap-heavy)
    (4, 256, 128, 17, None, None, None),              # L=17 taps
    (2, 64, 64, 1, None, 2, 1),                       # L=1: no kernel lags, only scale + background
    (2, 64, 8192, 3, None, 0, 0),                     # longest row FFT (W=8192), constant kernel
    (2, 64, 2048, 3, None, 1, 1),                     # W=2048 row FFT (radix 16-16-4)
    (3, 64, 4096, 5, None, 2, 1),                     # W=4096 row FFT (radix 16-16-8), the headline width
    (2, 128, 128, 9, None, 1, 2),                     # L without an exact subtract instantiation (padded taps)
    (2, 64, 1024, 9, None, 2, 1),                     # Fourier-route subtract (W >= 1024, L >= 9), 2w % 4 == 0
    (2, 256, 1024, 11, None, 1, 0),                   # Fourier route, 2w % 4 == 2 (padded lead-in), several x-ranges
    (3, 128, 2048, 15, None, 2, 2),                   # Fourier route, L = 15
    (4, 64, 4096, 17, None, 2, 2),                    # Fourier route at the headline width and kernel size
    (2, 128, 128, 33, None, 0, 0),                    # the largest kernel (L = 33: 65 lags per axis, 32-row hops)
    (2, 64, 1024, 25, None, 1, 1),                    # the widest kernel of the Fourier-route subtract (L = 25)
    (2, 128, 256, 27, None, 1, 0),                    # L = 27: direct subtract with 27 taps
    (5, 128, 128, 5, "bspline", 1, 0),                # B-spline weights
    (5, 256, 256, 5, "bspline", 4, 4),                # config-5 basis (8x8 functions), n = 1664
    # the edges of what sfft_plan_create accepts (DK, DB <= 8, H <= 8192)
    (2, 64, 128, 5, "poly", 4, 4),                    # 15 kernel terms: 16 column sequences on the direct lag sums
    (2, 64, 128, 3, "poly", 8, 8),                    # highest polynomial degree: 45 terms, 17 row moments per image
    (2, 128, 128, 3, "poly", 6, 6),                   # 13 row moments per image
    (5, 128, 128, 3, "bspline", 8, 8),                # most B-spline knots: 12 x 12 = 144 kernel terms, n = 1440
    (2, 8192, 64, 5, "poly", 1, 1),                   # tallest frame (H = 8192)
]


@pytest.mark.parametrize("cfg,H,W,L,basis,DK,DB", CASES)
def test_parity_small(cuda_device, cfg, H, W, L, basis, DK, DB):
    import torch
    p = synth.make_pair(cfg, H=H, W=W)
    L = p.L if L is None else L
    basis = p.basis if basis is None else basis
    DK = p.DK if DK is None else DK
    DB = p.DB if DB is None else DB
    Mo, ro, co, Do = _oracle_all(p.R, p.S, L, basis, DK, DB)
    M, rhs, c, D = _gpu_all(torch, p, L, basis, DK, DB)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, Mo.shape[0] - oracle.num_terms(_bid(basis), DB))
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


@pytest.mark.parametrize("cfg,H,W,L,DK,DB", [
    (1, None, None, None, None, None),      # config 1
    (3, 64, 256, 15, None, None),           # 29 lags on a small frame
    (4, 256, 128, 17, None, None),          # L = 17: lag-0 block + two 8-lag blocks
    (2, 128, 128, 9, 1, 2),
    (2, 64, 64, 1, 2, 1),                   # L = 1
])
def test_parity_direct_corr_route(cuda_device, cfg, H, W, L, DK, DB):
    """The polynomial cases take the sectioned FFT64 lag correlation by default; the direct tensor-core lag sums
    (the route of the many-term bases) must give the same system on the same input (sfft_plan_set_corr_route)."""
    import torch
    p = synth.make_pair(cfg, H=H, W=W)
    L = p.L if L is None else L
    DK = p.DK if DK is None else DK
    DB = p.DB if DB is None else DB
    Mo, ro, co, Do = _oracle_all(p.R, p.S, L, "poly", DK, DB)
    M, rhs, c, D = _gpu_all(torch, p, L, "poly", DK, DB, corr_route=1)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, Mo.shape[0] - oracle.num_terms(oracle.POLY, DB))
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


def test_parity_many_polynomial_terms_and_routes(cuda_device):
    """DK = 3: 10 kernel terms + S = 11 column sequences -> beyond the sectioned kernel's 8, the plan falls back to
    the direct lag sums by itself and refuses route 2; x-range splits of the sectioned route on a tall frame."""
    import torch
    p = synth.make_pair(2, H=128, W=128)
    Mo, ro, co, Do = _oracle_all(p.R, p.S, 5, "poly", 3, 1)
    M, rhs, c, D = _gpu_all(torch, p, 5, "poly", 3, 1)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    st, h = B.sfft_plan_create(128, 128, 5, 3, 1, 0)
    assert st == B.SFFT_OK and B.sfft_plan_set_corr_route(h, 2) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_plan_set_corr_route(h, 1) == B.SFFT_OK and B.sfft_plan_set_corr_route(h, 3) == B.SFFT_ERR_INVALID_ARG
    B.sfft_plan_destroy(h)
    p = synth.make_pair(2, H=2048, W=64)                       # few columns, many rows: the x axis is split in parts
    Mo, ro, co, Do = _oracle_all(p.R, p.S, 7, "poly", 2, 2)
    M, rhs, c, D = _gpu_all(torch, p, 7, "poly", 2, 2, corr_route=2)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, Mo.shape[0] - 6)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


def test_parity_config2_full(cuda_device):
    import torch
    p = synth.make_pair(2)
    Mo, ro, co, Do = _oracle_all(p.R, p.S, p.L, p.basis, p.DK, p.DB)
    M, rhs, c, D = _gpu_all(torch, p, p.L, p.basis, p.DK, p.DB)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, 6 * p.L * p.L)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


def _full_frame_both_modes(torch, p):
    """Full-size check shared by configs 3, 4 and the CCD frame: the oracle's full normal system, solution and FULL
    difference image (every pixel) against the CUDA path in both subtract modes -- the default, which transforms
    the reference again, and reuse_spectra=True, the launch configuration bench.py times (fit and apply on the same
    pair, the build's row spectra reused)."""
    bid = oracle.POLY
    Mo, ro = oracle.normal_from_lags(p.R, p.S, p.L, bid, p.DK, p.DB)
    co = oracle.solve(Mo, ro)
    Do = oracle.difference(p.R, p.S, co, p.L, bid, p.DK, p.DB)
    for reuse in (False, True):
        M, rhs, c, D = _gpu_all(torch, p, p.L, p.basis, p.DK, p.DB, reuse_spectra=reuse)
        _check_system(M[0], rhs[0], Mo, ro, p.S)
        _check_coef(c[0], co, 6 * p.L * p.L)
        assert D.shape == Do.shape and np.max(np.abs(D - Do)) <= TOL_D * p.sigma, f"reuse_spectra={reuse}"


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [3, 4])
def test_parity_full_size(cuda_device, cfg):
    """Configs 3 and 4 at BASELINE.json's full size: M, rhs, c and every pixel of D, in the default mode and in the
    launch configuration bench.py times (reuse_spectra=True).  The oracle's full direct-sum system takes about a
    minute or two of host time per config, its full difference image a few seconds."""
    import torch
    _full_frame_both_modes(torch, synth.make_pair(cfg))


@pytest.mark.slow
def test_parity_decam_ccd_frame_2046x4094(cuda_device):
    """NEXT-4 at the true DECam CCD size (2046 x 4094 = 2*3*11*31 x 2*23*89), config-3 recipe and model
    (15 x 15 delta basis, DK = DB = 2, n = 1356): full M / rhs / c element-wise, D on every pixel, both subtract modes."""
    import torch
    _full_frame_both_modes(torch, synth.make_pair(3, H=2046, W=4094))


@pytest.mark.slow
def test_parity_config5_batch64_in_one_call(cuda_device):
    """BASELINE.json configs[4] as stated: 64 independent 1024x1024 sub-field pairs (each seeded as in config 2),
    cubic B-splines with 4 interior knots per axis, 11x11 delta basis, n = 7808, processed in ONE call
    (nbatch = 64: batched row FFTs, the lag gather into 64 matrices of 488 MB, 64 concurrent solves on the
    throughput path).  Checked against the oracle as SURVEY 8(c) prescribes:
      * sub-fields 0 and 63: the oracle's FULL normal system (direct pixel sums), its solution and the full-frame
        difference -> M, rhs, c element by element, D on every pixel, at the g16 tolerances;
      * all 64: the diagonal of M and all of rhs against oracle.diag_and_rhs (column definitions), exact symmetry
        of M, the coefficients against the LAPACK + extended-precision-refined solution of the assembled system,
        and D at 600 pixels (corners included) through oracle.difference_at with that solution."""
    import os
    import scipy.linalg
    import torch
    nb = 64
    c5 = synth.CONFIGS[5]
    assert c5["batch"] == nb
    pb = synth.make_batch(5, workers=min(16, os.cpu_count() or 1))
    L, DK, DB, bid = c5["L"], c5["DK"], c5["DB"], oracle.BSPLINE
    plan = B.Plan(pb.H, pb.W, L, DK, DB, "bspline", nbatch=nb)
    dR, dS = torch.from_numpy(pb.R).cuda(), torch.from_numpy(pb.S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    dD = plan.subtract(coef, dR, dS)
    plan.status()
    c, D = coef.cpu().numpy(), dD.cpu().numpy()
    del dD, dR, dS
    n = plan.n
    na = n - oracle.num_terms(bid, DB)
    assert n == 7808 and c.shape == (nb, n)
    rng = np.random.default_rng(64)
    for e in range(nb):
        R, S = pb.R[e], pb.S[e]
        Mt, rt = plan.system(batch=e)
        M, rhs = Mt.cpu().numpy(), rt.cpu().numpy()
        del Mt, rt
        assert np.array_equal(M, M.T)
        dg, ro = oracle.diag_and_rhs(R, S, L, bid, DK, DB)
        d = np.sqrt(dg)
        assert np.max(np.abs(np.diag(M) - dg) / dg) <= TOL_M
        assert np.max(np.abs(rhs - ro) / (d * np.sqrt(np.sum(S * S)))) <= TOL_M
        if e in (0, nb - 1):
            Mo, ro2 = oracle.normal_from_lags(R, S, L, bid, DK, DB)
            co = oracle.solve(Mo, ro2)
            _check_system(M, rhs, Mo, ro2, S)
            _check_coef(c[e], co, na)
            Do = oracle.difference(R, S, co, L, bid, DK, DB)
            assert np.max(np.abs(D[e] - Do)) <= TOL_D * pb.sigma
            del Mo, Do
        # solution of the assembled system by LAPACK Cholesky + residuals in extended precision
        ds = 1.0 / np.sqrt(np.diag(M))
        Ms, rs = M * ds[:, None] * ds[None, :], rhs * ds
        cf = scipy.linalg.cho_factor(Ms, lower=True)
        x = scipy.linalg.cho_solve(cf, rs)
        r = rs.astype(np.longdouble) - Ms.astype(np.longdouble) @ x.astype(np.longdouble)
        x = x + scipy.linalg.cho_solve(cf, r.astype(np.float64))      # one refinement step: cond ~ 3e6
        del Ms
        cl = x * ds
        _check_coef(c[e], cl, na)
        px, py = rng.integers(0, pb.H, 600), rng.integers(0, pb.W, 600)
        px[:4], py[:4] = [0, 0, pb.H - 1, pb.H - 1], [0, pb.W - 1, 0, pb.W - 1]
        Dref = oracle.difference_at(R, S, cl, L, bid, DK, DB, px, py)
        assert np.max(np.abs(D[e][px, py] - Dref)) <= TOL_D * pb.sigma
    plan.close()


def test_batch_matches_single(cuda_device):
    """nbatch = 3 independent pairs in one call: each entry equals the oracle on that pair."""
    import torch
    pb = synth.make_batch(5, nbatch=3, H=128, W=128)
    L, DK, DB = 5, 1, 1
    M, rhs, c, D = _gpu_all(torch, pb, L, "bspline", DK, DB)
    for e in range(3):
        Mo, ro, co, Do = _oracle_all(pb.R[e], pb.S[e], L, "bspline", DK, DB)
        _check_system(M[e], rhs[e], Mo, ro, pb.S[e])
        _check_coef(c[e], co, Mo.shape[0] - 25)
        assert np.max(np.abs(D[e] - Do)) <= TOL_D * pb.sigma


def test_batch_solve_grid_beyond_one_wave(cuda_device):
    """nbatch = 5 systems of n = 1664: each factorisation launch holds ~1900 CTAs, several waves, so the
    panel CTAs of the later batch entries start after those of the first have finished (a write-back of
    the factored diagonal block would then be read as input by late CTAs).  Last entry against the
    oracle, every entry against the same pair run alone."""
    import torch
    nb, L, DK, DB = 5, 5, 4, 4
    pb = synth.make_batch(5, nbatch=nb, H=256, W=256)
    M, rhs, c, D = _gpu_all(torch, pb, L, "bspline", DK, DB)
    for e in range(nb):
        M1, r1, c1, D1 = _gpu_all(torch, pb, L, "bspline", DK, DB, R=pb.R[e], S=pb.S[e])
        assert np.max(np.abs(c[e] - c1[0])) <= TOL_C * np.max(np.abs(c1[0]))
        assert np.max(np.abs(D[e] - D1)) <= TOL_D * pb.sigma
    e = nb - 1
    Mo, ro, co, Do = _oracle_all(pb.R[e], pb.S[e], L, "bspline", DK, DB)
    _check_system(M[e], rhs[e], Mo, ro, pb.S[e])
    _check_coef(c[e], co, Mo.shape[0] - 64)
    assert np.max(np.abs(D[e] - Do)) <= TOL_D * pb.sigma


def test_batch_solve_large_batch_regime(cuda_device):
    """nbatch = 80 systems of n = 1664 (26 slabs): the solve takes its throughput path (one factoring CTA per
    system, lean slab CTAs, trailing update by tile rows with the cp.async double buffer).  Entries 0, 41, 79
    against the same pair run alone (latency path), entry 79 against the oracle."""
    import torch
    nb, L, DK, DB = 80, 5, 4, 4
    pb = synth.make_batch(5, nbatch=nb, H=128, W=128)
    M, rhs, c, D = _gpu_all(torch, pb, L, "bspline", DK, DB)
    for e in (0, 41, 79):
        M1, r1, c1, D1 = _gpu_all(torch, pb, L, "bspline", DK, DB, R=pb.R[e], S=pb.S[e])
        assert np.max(np.abs(c[e] - c1[0])) <= TOL_C * np.max(np.abs(c1[0]))
        assert np.max(np.abs(D[e] - D1)) <= TOL_D * pb.sigma
    e = nb - 1
    Mo, ro, co, Do = _oracle_all(pb.R[e], pb.S[e], L, "bspline", DK, DB)
    _check_coef(c[e], co, Mo.shape[0] - 64)
    assert np.max(np.abs(D[e] - Do)) <= TOL_D * pb.sigma


def test_batch_fourier_route(cuda_device):
    """nbatch = 2 through the Fourier-route subtract (per-entry kernel spectra and spectrum stacks)."""
    import torch
    pb = synth.make_batch(5, nbatch=2, H=64, W=1024)
    L, DK, DB = 9, 1, 1
    M, rhs, c, D = _gpu_all(torch, pb, L, "poly", DK, DB)
    for e in range(2):
        Mo, ro, co, Do = _oracle_all(pb.R[e], pb.S[e], L, "poly", DK, DB)
        _check_coef(c[e], co, Mo.shape[0] - 3)
        assert np.max(np.abs(D[e] - Do)) <= TOL_D * pb.sigma


@pytest.mark.parametrize("cfg,H,W,L,basis,DK,DB", [
    (1, None, None, None, "poly", 1, 1),          # config 1 with the paper's default -ConstPhotRatio True: 148 unknowns
    (2, 64, 1024, 9, "poly", 2, 1),               # Fourier-route subtract
    (5, 128, 128, 5, "bspline", 1, 0),            # B-splines: all centre coefficients equal (shared unknown sums 25 terms)
    (2, 64, 64, 1, "poly", 2, 1),                 # L = 1: only the scale and the background remain
])
def test_parity_constant_photometric_ratio(cuda_device, cfg, H, W, L, basis, DK, DB):
    """NEXT-1: constrained normal system, solution (full layout) and difference."""
    import torch
    p = synth.make_pair(cfg, H=H, W=W)
    L = p.L if L is None else L
    bid = _bid(basis)
    Mf, rf = oracle.normal_from_lags(p.R, p.S, L, bid, DK, DB)
    Mo, ro = oracle.cpr_constrain(Mf, rf, L, bid, DK, DB)
    co = oracle.cpr_expand(oracle.solve(Mo, ro), L, bid, DK, DB)
    Do = oracle.difference(p.R, p.S, co, L, bid, DK, DB)
    plan = B.Plan(p.H, p.W, L, DK, DB, basis, const_phot_ratio=True)
    assert plan.ns == oracle.cpr_num_unknowns(L, bid, DK, DB) and plan.n == Mf.shape[0]
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    plan.status()
    M, rhs = plan.system()
    _check_system(M[0].cpu().numpy(), rhs[0].cpu().numpy(), Mo, ro, p.S)
    _check_coef(coef[0].cpu().numpy(), co, Mf.shape[0] - oracle.num_terms(bid, DB))
    assert np.max(np.abs(D.cpu().numpy() - Do)) <= TOL_D * p.sigma
    plan.close()


@pytest.mark.parametrize("cfg,H,W,L,DK,DB", [
    (1, 96, 130, 7, 1, 1),        # neither axis a power of two; chirp-z rows with M = 512
    (2, 100, 1022, 5, 2, 1),      # W/2 = 511 = 7 x 73, M = 1024
    (2, 50, 4094, 3, 1, 1),       # the DECam row length 4094 = 2 x 23 x 89, M = 4096
    (3, 186, 372, 15, 2, 2),      # 2046 x 4094 scaled by 1/11: wide kernel, several hops and a ragged last one
    (2, 90, 1024, 5, 1, 1),       # only H is not a power of two (rows per CTA do not divide H)
    (2, 128, 1000, 9, 2, 0),      # only W is not a power of two
    (2, 100, 2046, 9, 2, 1),      # Fourier-route subtract on chirp-z rows (W/2 = 1023 >= 512, L >= 9): FIR with a ragged
                                  # last column block and x-range, inverse chirp-z transform
    (2, 90, 1024, 9, 1, 1),       # Fourier route, W a power of two, H not a multiple of the rows per CTA
    (3, 62, 4094, 15, 2, 2),      # Fourier route at the DECam row length, M = 4096
])
def test_parity_frames_not_powers_of_two(cuda_device, cfg, H, W, L, DK, DB):
    """NEXT-4 (true CCD frames such as 2046 x 4094): any H, even W - chirp-z row transforms, general
    wrap-around in the sectioned lag correlation, ragged tiles in the direct subtract."""
    import torch
    p = synth.make_pair(cfg, H=H, W=W)
    Mo, ro, co, Do = _oracle_all(p.R, p.S, L, "poly", DK, DB)
    M, rhs, c, D = _gpu_all(torch, p, L, "poly", DK, DB)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, Mo.shape[0] - oracle.num_terms(oracle.POLY, DB))
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


def test_combination_batch_rect_cpr_on_a_frame_not_a_power_of_two(cuda_device):
    """The section-8(f) options together: a batch of 2 pairs of 90 x 132 pixels, a 5 x 7 kernel, the constant
    photometric ratio; and the smallest frame the plan accepts (32 x 64)."""
    import torch
    L0, L1, DK, DB = 5, 7, 2, 1
    L = max(L0, L1)
    pairs = [synth.make_pair(2, H=90, W=132, seed=77 + e) for e in range(2)]
    R, S = np.stack([q.R for q in pairs]), np.stack([q.S for q in pairs])
    plan = B.Plan(90, 132, (L0, L1), DK, DB, "poly", nbatch=2, const_phot_ratio=True)
    dR, dS = torch.from_numpy(R).cuda(), torch.from_numpy(S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS).cpu().numpy()
    plan.status()
    FK, FB = oracle.num_terms(oracle.POLY, DK), oracle.num_terms(oracle.POLY, DB)
    a0 = ((L - 1) // 2) * L + (L - 1) // 2
    sel = oracle.rect_select(L0, L1, oracle.POLY, DK, DB)
    sel = np.array([k for k in sel if not (k < FK * L * L and k % (L * L) == a0 and k // (L * L) > 0)])
    assert plan.ns == len(sel)
    for e in range(2):
        Mf, rf = oracle.normal_from_lags(R[e], S[e], L, oracle.POLY, DK, DB)
        Mo, ro = Mf[np.ix_(sel, sel)], rf[sel]
        co = np.zeros(Mf.shape[0])
        co[sel] = oracle.solve(Mo, ro)
        M, rhs = plan.system(batch=e)
        _check_system(M.cpu().numpy(), rhs.cpu().numpy(), Mo, ro, S[e])
        _check_coef(coef[e].cpu().numpy(), co, Mf.shape[0] - FB)
        Do = oracle.difference(R[e], S[e], co, L, oracle.POLY, DK, DB)
        assert np.max(np.abs(D[e] - Do)) <= TOL_D * pairs[e].sigma
    plan.close()
    p = synth.make_pair(1, H=32, W=64)
    Mo, ro, co, Do = _oracle_all(p.R, p.S, 3, "poly", 1, 1)
    M, rhs, c, D = _gpu_all(torch, p, 3, "poly", 1, 1)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, Mo.shape[0] - 3)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


@pytest.mark.parametrize("cfg,H,W,L0,L1,basis,DK,DB,cpr", [
    (2, 128, 256, 5, 9, "poly", 2, 1, False),       # wider along y; direct-route subtract
    (2, 64, 1024, 13, 7, "poly", 1, 1, False),      # wider along x; Fourier-route subtract (W >= 1024, L = 13)
    (5, 128, 128, 3, 5, "bspline", 1, 0, False),    # B-spline weights, direct lag sums
    (2, 128, 128, 7, 3, "poly", 2, 2, True),        # together with the constant photometric ratio
    (2, 64, 64, 1, 5, "poly", 1, 1, False),         # a single column of lags (L0 = 1)
])
def test_parity_rectangular_kernel(cuda_device, cfg, H, W, L0, L1, basis, DK, DB, cpr):
    """NEXT-4 (the delta basis spans L0 x L1 pixels): system of the free unknowns, solution in the
    layout of the enclosing square (zeros outside the rectangle) and difference image, against the oracle's
    rectangular model (pinned to a direct L0 x L1 design matrix in tests/test_oracle_pins.py)."""
    import torch
    p = synth.make_pair(cfg, H=H, W=W)
    bid, L = _bid(basis), max(L0, L1)
    Mf, rf = oracle.normal_from_lags(p.R, p.S, L, bid, DK, DB)
    sel = oracle.rect_select(L0, L1, bid, DK, DB)
    FK, FB = oracle.num_terms(bid, DK), oracle.num_terms(bid, DB)
    if cpr:
        # constant kernel integral (POLY): the centre coefficients of the terms t >= 1 are zero as well
        a0 = ((L - 1) // 2) * L + (L - 1) // 2
        sel = np.array([k for k in sel if not (k < FK * L * L and k % (L * L) == a0 and k // (L * L) > 0)])
    Mo, ro = Mf[np.ix_(sel, sel)], rf[sel]
    cs = oracle.solve(Mo, ro)
    co = np.zeros(Mf.shape[0])
    co[sel] = cs
    Do = oracle.difference(p.R, p.S, co, L, bid, DK, DB)
    plan = B.Plan(p.H, p.W, (L0, L1), DK, DB, basis, const_phot_ratio=cpr)
    assert plan.n == Mf.shape[0] and plan.ns == len(sel) == FK * L0 * L1 + FB - (FK - 1 if cpr else 0)
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    plan.status()
    M, rhs = plan.system()
    _check_system(M[0].cpu().numpy(), rhs[0].cpu().numpy(), Mo, ro, p.S)
    c = coef[0].cpu().numpy()
    _check_coef(c, co, Mf.shape[0] - FB)
    fixed = np.setdiff1d(np.arange(Mf.shape[0]), sel)
    assert np.all(c[fixed] == 0.0)
    assert np.max(np.abs(D.cpu().numpy() - Do)) <= TOL_D * p.sigma
    plan.close()


def test_identical_images(cuda_device):
    """S = R  =>  a_{0,centre} = 1, everything else 0, D = 0 (degenerate but full-rank case)."""
    import torch
    p = synth.make_pair(1)
    M, rhs, c, D = _gpu_all(torch, p, 5, "poly", 1, 1, R=p.R, S=p.R.copy())
    e = np.zeros_like(c[0]); e[12] = 1.0
    assert np.max(np.abs(c[0] - e)) <= 1e-9
    assert np.max(np.abs(D)) <= TOL_D * p.sigma


@pytest.mark.parametrize("H,W,L", [(None, None, None), (64, 1024, 9)])
def test_fit_on_one_pair_apply_to_another_and_inplace(cuda_device, H, W, L):
    """solve on the masked pair, apply to the original pair; D may alias S.
    The second shape takes the Fourier-route subtract, which must transform the new R itself
    (the row spectra cached by build belong to the masked reference)."""
    import torch
    p = synth.make_pair(1, H=H, W=W)
    p.L = p.L if L is None else L
    mask = np.ones_like(p.R); mask[40:60, 30:50] = 0.0
    Rm, Sm = p.R * mask + 100.0 * (1 - mask), p.S * mask + 100.0 * (1 - mask)
    Mo, ro = oracle.normal_from_lags(Rm, Sm, p.L, oracle.POLY, p.DK, p.DB)
    co = oracle.solve(Mo, ro)
    Do = oracle.difference(p.R, p.S, co, p.L, oracle.POLY, p.DK, p.DB)
    plan = B.Plan(p.H, p.W, p.L, p.DK, p.DB, "poly")
    plan.build_system(torch.from_numpy(Rm).cuda(), torch.from_numpy(Sm).cuda())
    coef = plan.solve()
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    out = plan.subtract(coef, dR, dS, D=dS)      # in place
    plan.status()
    assert out.data_ptr() == dS.data_ptr()
    assert np.max(np.abs(dS.cpu().numpy() - Do)) <= TOL_D * p.sigma
    plan.close()


def test_subtract_after_address_reuse_and_inplace_edit(cuda_device):
    """The masked flow of PAPER.md:218 under a caching allocator: the masked reference is freed after the build
    and the ORIGINAL reference lands at the very same device address.  The Fourier-route subtract must transform
    the buffer it is given (default contract: no reuse of the build's spectra, whatever the pointers are), and
    the same when the fitted buffer is edited in place (un-masked) between build and subtract."""
    import torch
    p = synth.make_pair(1, H=64, W=1024)
    L = 9
    mask = np.ones_like(p.R); mask[20:40, 300:420] = 0.0
    Rm, Sm = p.R * mask + 100.0 * (1 - mask), p.S * mask + 100.0 * (1 - mask)
    Mo, ro = oracle.normal_from_lags(Rm, Sm, L, oracle.POLY, p.DK, p.DB)
    co = oracle.solve(Mo, ro)
    Do = oracle.difference(p.R, p.S, co, L, oracle.POLY, p.DK, p.DB)
    plan = B.Plan(p.H, p.W, L, p.DK, p.DB, "poly")
    dS, dSm = torch.from_numpy(p.S).cuda(), torch.from_numpy(Sm).cuda()
    coef = torch.empty((1, plan.n), dtype=torch.float64, device="cuda")
    hit = False
    for _ in range(50):                       # until the allocator hands the freed block back
        dRm = torch.from_numpy(Rm).cuda()
        addr = dRm.data_ptr()
        plan.build_system(dRm, dSm)
        plan.solve(coef)
        torch.cuda.synchronize()
        del dRm
        dR = torch.from_numpy(p.R).cuda()
        if dR.data_ptr() == addr:
            hit = True
            break
        del dR
    assert hit, "the caching allocator never reused the freed block"
    D = plan.subtract(coef, dR, dS)
    plan.status()
    assert np.max(np.abs(D.cpu().numpy() - Do)) <= TOL_D * p.sigma
    # in-place edit of the fitted buffer
    dX = torch.from_numpy(Rm).cuda()
    plan.build_system(dX, dSm)
    plan.solve(coef)
    dX.copy_(torch.from_numpy(p.R))
    D = plan.subtract(coef, dX, dS)
    plan.status()
    assert np.max(np.abs(D.cpu().numpy() - Do)) <= TOL_D * p.sigma
    # the opt-in reuse (same pair for fit and apply) gives the same difference as the default on that pair
    Dm0 = plan.subtract(coef, dX, dS).cpu().numpy()
    plan2 = B.Plan(p.H, p.W, L, p.DK, p.DB, "poly", reuse_spectra=True)
    plan2.build_system(dX, dS)
    c2 = plan2.solve()
    D2 = plan2.subtract(c2, dX, dS)
    D2b = plan2.subtract(c2, dX, dS)          # second subtract after the same build: spectra still valid
    plan2.status()
    _, _, co2, Do2 = _oracle_all(p.R, p.S, L, "poly", p.DK, p.DB)
    assert np.max(np.abs(D2.cpu().numpy() - Do2)) <= TOL_D * p.sigma
    assert np.array_equal(D2.cpu().numpy(), D2b.cpu().numpy())
    assert Dm0.shape == Do.shape
    plan.close(); plan2.close()


def _saturate(p, sat, nsat=12, seed=5):
    """Clip the brightest stars of a pair at `sat` plus a few bleed columns, as saturated sources look on a CCD."""
    rng = np.random.default_rng(seed)
    R, S = p.R.copy(), p.S.copy()
    idx = np.argsort(R.ravel())[-nsat:]
    for q in idx:
        x, y = divmod(int(q), p.W)
        h = int(rng.integers(2, 6))
        for dx in range(-h, h + 1):
            R[(x + dx) % p.H, y] = sat * 1.2
            S[(x + dx) % p.H, y] = sat * 1.1
    R[0, 0] = sat * 2; S[p.H - 1, p.W - 1] = sat * 3          # corners: the window wraps around the frame
    return np.minimum(R, sat * 4), np.minimum(S, sat * 4)


@pytest.mark.parametrize("cfg,H,W,L,rd,rb,nb", [(1, None, None, None, 2, 6, 1), (2, 64, 1024, 9, 1, 4, 1), (5, 128, 128, 5, 3, 8, 3),
                                                 (1, 96, 130, 7, 2, 6, 1)])
def test_mask_fill_and_masked_fit_flow(cuda_device, cfg, H, W, L, rd, rb, nb):
    """NEXT-2 (DESIGN g21): the CUDA mask/fill against the oracle (mask bit-exact, filled pixels to
    rounding), then the paper's two-step flow end to end: fit on the masked pair, apply to the original pair."""
    import torch
    sat = 3000.0
    if nb == 1:
        p = synth.make_pair(cfg, H=H, W=W)
        Rs, Ss = _saturate(p, sat)
        Rl, Sl = [Rs], [Ss]
    else:
        p = synth.make_batch(cfg, nbatch=nb, H=H, W=W)
        pp = [synth.Pair(R=p.R[e], S=p.S[e], H=p.H, W=p.W, L=p.L, DK=1, DB=1, basis="poly", sigma=p.sigma, config=cfg) for e in range(nb)]
        Rl, Sl = zip(*[_saturate(q, sat, seed=e) for e, q in enumerate(pp)])
        Rs, Ss = np.stack(Rl), np.stack(Sl)
    L = p.L if L is None else L
    DK, DB, basis = (p.DK, p.DB, p.basis) if nb == 1 else (1, 1, "poly")
    plan = B.Plan(p.H, p.W, L, DK, DB, basis, nbatch=nb)
    dR, dS = torch.from_numpy(np.ascontiguousarray(Rs)).cuda(), torch.from_numpy(np.ascontiguousarray(Ss)).cuda()
    dRm, dSm, dmask = plan.mask_fill(dR, dS, sat, sat, rd, rb)
    plan.build_system(dRm, dSm)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    plan.status()
    Rm, Sm, mask = dRm.cpu().numpy().reshape(nb, p.H, p.W), dSm.cpu().numpy().reshape(nb, p.H, p.W), dmask.cpu().numpy().reshape(nb, p.H, p.W)
    c, D = coef.cpu().numpy(), D.cpu().numpy().reshape(nb, p.H, p.W)
    bid = _bid(basis)
    for e in range(nb):
        Rmo, Smo, mo = oracle.mask_fill(Rl[e], Sl[e], sat, sat, rd, rb)
        assert mo.sum() > 0 and np.array_equal(mask[e], mo)
        assert np.max(np.abs(Rm[e] - Rmo)) <= 1e-12 * sat and np.max(np.abs(Sm[e] - Smo)) <= 1e-12 * sat
        assert np.array_equal(Rm[e][mo == 0], Rl[e][mo == 0])
        Mo, ro = oracle.normal_from_lags(Rmo, Smo, L, bid, DK, DB)
        co = oracle.solve(Mo, ro)
        Do = oracle.difference(Rl[e], Sl[e], co, L, bid, DK, DB)
        _check_coef(c[e], co, Mo.shape[0] - oracle.num_terms(bid, DB))
        assert np.max(np.abs(D[e] - Do)) <= TOL_D * p.sigma
    # in place, and argument errors
    dR2, dS2 = dR.clone(), dS.clone()
    a, b_, m2 = plan.mask_fill(dR2, dS2, sat, sat, rd, rb, inplace=True)
    assert a.data_ptr() == dR2.data_ptr() and torch.equal(dR2, dRm) and torch.equal(dS2, dSm) and torch.equal(m2, dmask)
    assert B.sfft_mask_fill(plan.h, dR.data_ptr(), dS.data_ptr(), sat, sat, -1, rb, dRm.data_ptr(), dSm.data_ptr(), dmask.data_ptr()) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_mask_fill(plan.h, dR.data_ptr(), dS.data_ptr(), sat, sat, rd, 0, dRm.data_ptr(), dSm.data_ptr(), dmask.data_ptr()) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_mask_fill(plan.h, dR.data_ptr(), 0, sat, sat, rd, rb, dRm.data_ptr(), dSm.data_ptr(), dmask.data_ptr()) == B.SFFT_ERR_INVALID_ARG
    plan.close()


@pytest.mark.parametrize("cfg,H,W,L,DK,tile,coadd", [(1, 128, 128, 7, 1, 32, False), (2, 256, 512, 11, 2, 128, True),
                                                        (2, 512, 512, 9, 2, 512, False), (2, 64, 1024, 5, 0, 64, True),
                                                        (1, 96, 160, 7, 1, 32, False)])
def test_decorrelation_parity(cuda_device, cfg, H, W, L, DK, tile, coadd):
    """NEXT-3 (App. C, Eq. C20; DESIGN g22): fit, subtract, then decorrelate on the GPU; the oracle decorrelates the
    GPU's difference image with the GPU's coefficients (both already checked against the oracle elsewhere), so this
    compares the decorrelation step alone, tile by tile, including the spatially varying kernel frozen at the tile
    centres and co-addition kernels G_j, H_i."""
    import torch
    from oracle import decorr
    p = synth.make_pair(cfg, H=H, W=W)
    DB = 1
    plan = B.Plan(H, W, L, DK, DB, "poly")
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    if coadd:
        g = np.array([[0.0, 0.1, 0.0], [0.1, 0.6, 0.1], [0.0, 0.1, 0.0]])
        var_S, G = [120.0, 130.0], np.stack([g / 2, np.roll(g, 1, axis=1) / 2])
        hk = np.zeros((5, 5)); hk[2, 2] = 0.5; hk[1, 2] = hk[3, 2] = 0.2; hk[2, 0] = 0.1
        var_R, Hk = [125.0, 110.0, 140.0], np.stack([hk / 3, hk.T / 3, hk[::-1] / 3])
    else:
        var_S, G, var_R, Hk = [125.0], np.ones((1, 1, 1)), [125.0], np.ones((1, 1, 1))
    Ddc = plan.decorrelate(coef, D, tile, var_S, G, var_R, Hk)
    plan.status()
    Dn, cn = D.cpu().numpy(), coef.cpu().numpy()[0]
    ref = decorr.decorrelate(Dn, cn, L, oracle.POLY, DK, tile, var_S, G, var_R, Hk)
    assert np.max(np.abs(ref - Dn)) > 1e-3 * p.sigma                       # the step does something
    assert np.max(np.abs(Ddc.cpu().numpy() - ref)) <= TOL_D * p.sigma
    # in place, and the documented argument errors
    D2 = D.clone()
    plan.decorrelate(coef, D2, tile, var_S, G, var_R, Hk, out=D2)
    plan.status()
    assert torch.equal(D2, Ddc)
    for bad_tile in (48, 16, 1024):
        assert B.sfft_decorrelate(plan.h, coef.data_ptr(), D.data_ptr(), D2.data_ptr(), bad_tile, var_S, G, var_R, Hk) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_decorrelate(plan.h, coef.data_ptr(), D.data_ptr(), D2.data_ptr(), tile, var_S, np.ones((len(var_S), 2, 2)), var_R, Hk) == B.SFFT_ERR_INVALID_ARG
    plan.close()


@pytest.mark.parametrize("cfg,H,W,L,DK,tile", [(1, 128, 128, 7, 1, 32), (2, 256, 512, 9, 2, 128)])
def test_decorrelation_chained_from_the_oracle_fit(cuda_device, cfg, H, W, L, DK, tile):
    """The whole chain on each side, nothing handed across: oracle fit -> oracle D -> oracle decorrelation against
    GPU build -> solve -> subtract -> sfft_decorrelate.  Tolerance: the decorrelated image is D convolved with a
    unit-sum kernel Q whose taps depend smoothly on the fitted kernel, so the 1e-6 sigma allowed on D and the 1e-8
    relative allowed on the coefficients carry through with a factor sum|Q| of order one: 4e-6 sigma."""
    import torch
    from oracle import decorr
    p = synth.make_pair(cfg, H=H, W=W)
    DB = 1
    _, _, co, Do = _oracle_all(p.R, p.S, L, "poly", DK, DB)
    g = np.array([[0.0, 0.1, 0.0], [0.1, 0.6, 0.1], [0.0, 0.1, 0.0]])
    var_S, G, var_R, Hk = [120.0, 130.0], np.stack([g / 2, np.roll(g, 1, axis=1) / 2]), [125.0], np.ones((1, 1, 1))
    ref = decorr.decorrelate(Do, co, L, oracle.POLY, DK, tile, var_S, G, var_R, Hk)
    plan = B.Plan(H, W, L, DK, DB, "poly")
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    plan.build_system(dR, dS)
    coef = plan.solve()
    D = plan.subtract(coef, dR, dS)
    Ddc = plan.decorrelate(coef, D, tile, var_S, G, var_R, Hk)
    plan.status()
    assert np.max(np.abs(ref - Do)) > 1e-3 * p.sigma
    assert np.max(np.abs(Ddc.cpu().numpy().reshape(H, W) - ref)) <= 4 * TOL_D * p.sigma
    plan.close()


def test_run_host_end_to_end(cuda_device):
    p = synth.make_pair(1)
    _, _, co, Do = _oracle_all(p.R, p.S, p.L, p.basis, p.DK, p.DB)
    plan = B.Plan(p.H, p.W, p.L, p.DK, p.DB, p.basis)
    D, c = plan.run_host(p.R, p.S)
    _check_coef(c[0], co, 3 * p.L * p.L)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma
    assert plan.launch_count() > 0
    plan.close()


def test_run_host_f32_storage(cuda_device):
    """NEXT-4: images stored as float on the host, arithmetic in FP64.  The oracle gets the same float-rounded
    images (exactly representable in double); coefficients at the usual tolerance; D equals the oracle's D up to the
    one rounding to float on the way out (half an ulp of float at |D|) plus the usual 1e-6 sigma."""
    import torch
    p = synth.make_pair(2, H=64, W=1024)
    L = 9
    R32, S32 = p.R.astype(np.float32), p.S.astype(np.float32)
    _, _, co, Do = _oracle_all(R32.astype(np.float64), S32.astype(np.float64), L, "poly", p.DK, p.DB)
    plan = B.Plan(p.H, p.W, L, p.DK, p.DB, "poly")
    D, c = plan.run_host(R32, S32)
    assert D.dtype == np.float32
    _check_coef(c[0], co, 6 * L * L)
    tol = TOL_D * p.sigma + np.abs(Do) * 2.0 ** -24 * 1.0001
    assert np.all(np.abs(D.astype(np.float64) - Do) <= tol)
    # mixed traffic through the two staging slots: f32, f64, f32 back to back, one wait
    hR, hS = torch.from_numpy(R32).pin_memory(), torch.from_numpy(S32).pin_memory()
    hR64, hS64 = torch.from_numpy(p.R).pin_memory(), torch.from_numpy(p.S).pin_memory()
    hD = [torch.empty_like(hR).pin_memory(), torch.empty_like(hR64).pin_memory(), torch.empty_like(hR).pin_memory()]
    hC = [torch.empty((1, plan.n), dtype=torch.float64).pin_memory() for _ in range(3)]
    assert B.sfft_run_host_async_f32(plan.h, hR.data_ptr(), hS.data_ptr(), hD[0].data_ptr(), hC[0].data_ptr()) == B.SFFT_OK
    assert B.sfft_run_host_async(plan.h, hR64.data_ptr(), hS64.data_ptr(), hD[1].data_ptr(), hC[1].data_ptr()) == B.SFFT_OK
    assert B.sfft_run_host_async_f32(plan.h, hR.data_ptr(), hS.data_ptr(), hD[2].data_ptr(), hC[2].data_ptr()) == B.SFFT_OK
    assert B.sfft_run_host_wait(plan.h) == B.SFFT_OK
    assert np.array_equal(hD[0].numpy(), D) and np.array_equal(hD[2].numpy(), D) and np.array_equal(hC[2].numpy(), c)
    _, _, co64, Do64 = _oracle_all(p.R, p.S, L, "poly", p.DK, p.DB)
    assert np.max(np.abs(hD[1].numpy() - Do64)) <= TOL_D * p.sigma
    plan.close()


def test_run_host_async_pipeline(cuda_device):
    """Three different pairs submitted back to back through sfft_run_host_async (two staging slots, copy streams):
    every result equals the one-call-at-a-time result of that pair."""
    import torch
    ps = [synth.make_pair(1, seed=900 + i) for i in range(3)]
    plan = B.Plan(ps[0].H, ps[0].W, ps[0].L, ps[0].DK, ps[0].DB, ps[0].basis)
    assert B.sfft_run_host_async(plan.h, 1, 1, 0, 0) == B.SFFT_ERR_WORKSPACE      # no staging area lent yet
    ref = [plan.run_host(p.R, p.S) for p in ps]
    hR = [torch.from_numpy(p.R).pin_memory() for p in ps]
    hS = [torch.from_numpy(p.S).pin_memory() for p in ps]
    hD = [torch.empty_like(x).pin_memory() for x in hR]
    hC = [torch.empty((1, plan.n), dtype=torch.float64).pin_memory() for _ in ps]
    for i in range(3):
        assert B.sfft_run_host_async(plan.h, hR[i].data_ptr(), hS[i].data_ptr(), hD[i].data_ptr(), hC[i].data_ptr()) == B.SFFT_OK
    assert B.sfft_run_host_wait(plan.h) == B.SFFT_OK
    for i in range(3):
        assert np.array_equal(hD[i].numpy(), ref[i][0])
        assert np.array_equal(hC[i].numpy(), ref[i][1])
    _, _, co, Do = _oracle_all(ps[2].R, ps[2].S, ps[2].L, ps[2].basis, ps[2].DK, ps[2].DB)
    assert np.max(np.abs(hD[2].numpy() - Do)) <= TOL_D * ps[2].sigma
    plan.close()


def test_rank_deficient_input_reports_not_spd(cuda_device):
    """DESIGN g11: a constant reference makes the shifted-difference columns vanish -> M singular."""
    import torch
    plan = B.Plan(64, 64, 3, 0, 0, "poly")
    R = torch.full((64, 64), 100.0, dtype=torch.float64, device="cuda")
    S = torch.rand((64, 64), dtype=torch.float64, device="cuda")
    plan.build_system(R, S)
    plan.solve()
    st, info = plan.status(check=False)
    assert st == B.SFFT_ERR_NOT_SPD and 0 <= info < plan.n
    plan.close()


def test_numerically_rank_deficient_input_reports_not_spd(cuda_device):
    """A reference made of one sine wave along y plus a constant: the 2w shifted-difference columns of a row of
    lags span only two functions (sin, cos), so M is singular, but its FFT-assembled entries carry rounding
    noise and the vanishing pivots come out as +-1e-16-sized numbers of either sign.  The pivot floor
    (64 n eps on the unit-diagonal scaled matrix) must flag them instead of returning garbage with SFFT_OK."""
    import torch
    H = W = 64
    y = np.arange(W)[None, :] * np.ones((H, 1))
    x = np.arange(H)[:, None] * np.ones((1, W))
    R = 100.0 + 10.0 * np.sin(2 * np.pi * y / W) + 5.0 * np.cos(2 * np.pi * x / H)
    rng = np.random.default_rng(3)
    S = R + rng.normal(0.0, 1.0, R.shape)
    plan = B.Plan(H, W, 5, 0, 0, "poly")
    plan.build_system(torch.from_numpy(R).cuda(), torch.from_numpy(S).cuda())
    plan.solve()
    st, info = plan.status(check=False)
    assert st == B.SFFT_ERR_NOT_SPD and 0 <= info < plan.n
    plan.close()


@pytest.mark.timeout(300)
def test_nan_input_with_sentinel_payload_does_not_stall_the_back_substitution(cuda_device):
    """The look-back back substitution marks "block not yet published" with a NaN bit pattern.  A NaN of that very payload
    in the input propagates through the arithmetic: the solve must still terminate and report SFFT_ERR_NOT_SPD."""
    import struct
    import torch
    p = synth.make_pair(1)
    R = p.R.copy()
    R[17, 23] = struct.unpack("<d", struct.pack("<Q", 0xFFF8DEADBEEF5AFE))[0]
    plan = B.Plan(p.H, p.W, p.L, p.DK, p.DB, p.basis)
    dR, dS = torch.from_numpy(R).cuda(), torch.from_numpy(p.S).cuda()
    plan.build_system(dR, dS)
    plan.solve()
    st, _ = plan.status(check=False)
    assert st == B.SFFT_ERR_NOT_SPD
    plan.close()


def test_step_is_capturable_in_a_cuda_graph(cuda_device):
    """build -> solve -> subtract captured once in a CUDA graph (side-stream fork / join of the moment stage,
    programmatic dependent launches of the panel chain, TMA tile copies of the back substitution) and replayed on
    new contents of the same buffers gives the result of the direct calls."""
    import torch
    p = synth.make_pair(2, H=128, W=1024)
    q = synth.make_pair(2, H=128, W=1024, seed=5)
    plan = B.Plan(p.H, p.W, 9, 2, 1, "poly")
    dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
    dD = torch.empty_like(dS)
    coef = torch.empty((1, plan.n), dtype=torch.float64, device="cuda")

    def step():
        plan.build_system(dR, dS)
        plan.solve(coef)
        plan.subtract(coef, dR, dS, dD)

    step()
    plan.status()
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        B.sfft_plan_set_stream(plan.h, s.cuda_stream)
        step()
        torch.cuda.synchronize()
        g.capture_begin()
        step()
        g.capture_end()
    torch.cuda.synchronize()
    dR.copy_(torch.from_numpy(q.R))
    dS.copy_(torch.from_numpy(q.S))
    g.replay()
    torch.cuda.synchronize()
    Dg, cg = dD.clone(), coef.clone()
    B.sfft_plan_set_stream(plan.h, plan.stream.cuda_stream)
    step()
    plan.status()
    assert torch.equal(dD, Dg) and torch.equal(coef, cg)
    Mo, ro, co, Do = _oracle_all(q.R, q.S, 9, "poly", 2, 1)
    assert np.max(np.abs(Dg.cpu().numpy() - Do)) <= TOL_D * q.sigma
    plan.close()


def test_argument_and_state_errors(cuda_device):
    import torch
    for bad in [(100, 129, 7, 1, 1, 0), (100, 4100, 7, 1, 1, 0), (100, 130, 7, 1, 1, 1), (100, 130, 7, 3, 1, 0), (128, 128, 6, 1, 1, 0), (128, 128, 7, -1, 1, 0), (128, 128, 7, 1, 1, 2),
                (64, 64, 33, 1, 1, 0), (16, 128, 3, 1, 1, 0)]:
        st, _ = B.sfft_plan_create(*bad)
        assert st == B.SFFT_ERR_INVALID_ARG, bad
    for bad in [(128, 128, 4, 7, 1, 1, 0), (128, 128, 7, 35, 1, 1, 0), (64, 64, 3, 33, 1, 1, 0), (128, 128, 0, 3, 1, 1, 0)]:
        st, _ = B.sfft_plan_create_rect(*bad)
        assert st == B.SFFT_ERR_INVALID_ARG, bad
    st, h = B.sfft_plan_create_rect(128, 128, 3, 7, 1, 1, 0)
    assert st == B.SFFT_OK and B.sfft_plan_num_unknowns(h) == 150 and B.sfft_plan_num_solved(h) == 3 * 21 + 3
    B.sfft_plan_destroy(h)
    st, h = B.sfft_plan_create(128, 128, 7, 1, 1, 0)
    assert st == B.SFFT_OK and B.sfft_plan_num_unknowns(h) == 150
    x = torch.zeros(128 * 128, dtype=torch.float64, device="cuda")
    assert B.sfft_build_system(h, x.data_ptr(), x.data_ptr()) == B.SFFT_ERR_WORKSPACE
    ws = torch.empty(B.sfft_plan_workspace_bytes(h) + 256, dtype=torch.uint8, device="cuda")
    ptr = (ws.data_ptr() + 255) & ~255
    assert B.sfft_plan_set_workspace(h, ptr, 1024) == B.SFFT_ERR_WORKSPACE
    assert B.sfft_plan_set_workspace(h, ptr, B.sfft_plan_workspace_bytes(h)) == B.SFFT_OK
    assert B.sfft_solve(h, x.data_ptr()) == B.SFFT_ERR_STATE
    assert B.sfft_build_system(h, 0, x.data_ptr()) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_plan_set_const_phot_ratio(h, 2) == B.SFFT_ERR_INVALID_ARG
    assert B.sfft_plan_set_const_phot_ratio(h, 1) == B.SFFT_OK and B.sfft_plan_num_solved(h) == 148
    assert B.sfft_plan_num_unknowns(h) == 150                      # coefficient vectors keep the full layout
    assert B.sfft_plan_set_const_phot_ratio(h, 0) == B.SFFT_OK and B.sfft_plan_num_solved(h) == 150
    assert B.sfft_run_host_async(h, 0, x.data_ptr(), 0, 0) == B.SFFT_ERR_INVALID_ARG
    st2, h2 = B.sfft_plan_create(128, 128, 7, 1, 1, 0)
    assert B.sfft_run_host_async(h2, x.data_ptr(), x.data_ptr(), 0, 0) == B.SFFT_ERR_WORKSPACE
    B.sfft_plan_destroy(h2)
    B.sfft_plan_destroy(h)


def test_stage_profile_splits_the_fourier_route_subtract(cuda_device):
    """sfft_plan_profile / sfft_plan_profile_read: every stage of a step gets a time; on the Fourier-route subtract
    stage 7 is the sum of its two parts (8 FIR along x, 9 inverse rows + difference), on the direct route the two
    parts read -1."""
    import torch
    for (H, W, L, fourier) in [(64, 1024, 9, True), (128, 128, 7, False)]:
        p = synth.make_pair(2, H=H, W=W)
        plan = B.Plan(H, W, L, 1, 1, "poly")
        dR, dS = torch.from_numpy(p.R).cuda(), torch.from_numpy(p.S).cuda()
        plan.profile(2)
        for _ in range(2):
            plan.build_system(dR, dS)
            coef = plan.solve()
            plan.subtract(coef, dR, dS)
        ms = plan.profile_read(2)
        plan.status()
        assert ms.shape == (2, B.SFFT_NUM_STAGES) and len(B.STAGE_NAMES) == B.SFFT_NUM_STAGES
        assert np.all(ms[:, :8] > 0.0)
        if fourier:
            assert np.all(ms[:, 8:] > 0.0) and np.allclose(ms[:, 8] + ms[:, 9], ms[:, 7], rtol=0.05, atol=2e-3)
        else:
            assert np.all(ms[:, 8:] == -1.0)
        plan.close()
