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
from paper_2109_09334_b200 import synth

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


def _gpu_all(torch, p, L, basis, DK, DB, R=None, S=None):
    R = p.R if R is None else R
    S = p.S if S is None else S
    nb = 1 if R.ndim == 2 else R.shape[0]
    H, W = R.shape[-2:]
    plan = B.Plan(H, W, L, DK, DB, basis, nbatch=nb)
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
    (5, 128, 128, 5, "bspline", 1, 0),                # B-spline weights
    (5, 256, 256, 5, "bspline", 4, 4),                # config-5 basis (8x8 functions), n = 1664
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


def test_parity_config2_full(cuda_device):
    import torch
    p = synth.make_pair(2)
    Mo, ro, co, Do = _oracle_all(p.R, p.S, p.L, p.basis, p.DK, p.DB)
    M, rhs, c, D = _gpu_all(torch, p, p.L, p.basis, p.DK, p.DB)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, 6 * p.L * p.L)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [3, 4])
def test_parity_full_size(cuda_device, cfg):
    """Configs 3 and 4 at BASELINE.json's full size, in the launch configuration bench.py times.
    The oracle's full direct-sum system takes about a minute or two of host time per config."""
    import torch
    p = synth.make_pair(cfg)
    bid = oracle.POLY
    Mo, ro = oracle.normal_from_lags(p.R, p.S, p.L, bid, p.DK, p.DB)
    co = oracle.solve(Mo, ro)
    M, rhs, c, D = _gpu_all(torch, p, p.L, p.basis, p.DK, p.DB)
    _check_system(M[0], rhs[0], Mo, ro, p.S)
    _check_coef(c[0], co, 6 * p.L * p.L)
    rng = np.random.default_rng(cfg)
    px = np.r_[rng.integers(0, p.H, 4000), [0, 0, p.H - 1, p.H - 1, 3, p.H - 2]]       # random + corners/borders
    py = np.r_[rng.integers(0, p.W, 4000), [0, p.W - 1, 0, p.W - 1, p.W - 4, 5]]
    Dref = oracle.difference_at(p.R, p.S, co, p.L, bid, p.DK, p.DB, px, py)
    assert np.max(np.abs(D[px, py] - Dref)) <= TOL_D * p.sigma


def _oracle_column(R, L, bid, DK, DB, k, wcache):
    """Column k of the design matrix Phi (Eqs. 3-4, 11-12) from the oracle's weighted images / axis tables."""
    H, W = R.shape
    LL, w = L * L, (L - 1) // 2
    FK = oracle.num_terms(bid, DK)
    if k < FK * LL:
        t, a = divmod(k, LL)
        al, be = a // L - w, a % L - w
        if t not in wcache:
            wcache[t] = oracle.weighted_ref(R, bid, DK, t)
        Rt = wcache[t]
        return Rt if (al == 0 and be == 0) else np.roll(Rt, (al, be), axis=(0, 1)) - Rt
    i, j = oracle.terms(bid, DB)[k - FK * LL]
    return np.outer(oracle.axis_table(bid, H, DB)[i], oracle.axis_table(bid, W, DB)[j])


@pytest.mark.slow
def test_parity_config5_full_size(cuda_device):
    """Config 5 at BASELINE.json's sub-field size and basis (1024x1024, L=11, cubic B-splines with 4 interior
    knots per axis, n = 7808), two sub-fields in one batched call.  The oracle's full system for this case is
    ~1e12 pixel sums plus an unblocked n=7808 factorisation per sub-field, so it is checked on sampled outputs
    the oracle computes one by one: 150 entries of M and 40 of rhs from the definition (oracle-weighted images,
    np.roll), D on 2000 pixels through oracle.difference_at, and the coefficients against LAPACK + long-double
    iterative refinement applied to the (sample-checked) GPU matrix."""
    import torch
    nb = 2
    c5 = synth.CONFIGS[5]
    pb = synth.make_batch(5, nbatch=nb)
    L, DK, DB, bid = c5["L"], c5["DK"], c5["DB"], oracle.BSPLINE
    M, rhs, c, D = _gpu_all(torch, pb, L, "bspline", DK, DB)
    n = M.shape[1]
    na = n - oracle.num_terms(bid, DB)
    assert n == 7808
    rng = np.random.default_rng(55)
    for e in range(nb):
        R, S = pb.R[e], pb.S[e]
        assert np.array_equal(M[e], M[e].T)
        d = np.sqrt(np.diag(M[e]))
        # sampled entries: neighbouring spatial terms and lags (large), far-apart terms (zero overlap), background
        ks = np.r_[rng.integers(0, na, 24), rng.integers(na, n, 6), [0, 60, na - 1, n - 1]]
        cols, wc = {}, {}
        for k in ks:
            cols[int(k)] = _oracle_column(R, L, bid, DK, DB, int(k), wc)
        kk = list(cols)
        worst = 0.0
        for a in range(len(kk)):
            for b in range(a, len(kk), 3):
                ref = float(np.sum(cols[kk[a]].astype(np.longdouble) * cols[kk[b]]))
                worst = max(worst, abs(M[e][kk[a], kk[b]] - ref) / (d[kk[a]] * d[kk[b]]))
        assert worst <= TOL_M, worst
        sn = np.sqrt(np.sum(S * S))
        for k in kk:
            ref = float(np.sum(cols[k].astype(np.longdouble) * S))
            assert abs(rhs[e][k] - ref) <= TOL_M * d[k] * sn
        # solution of the GPU's own system by LAPACK + extended-precision refinement
        ds = 1.0 / d
        Ms, rs = M[e] * ds[:, None] * ds[None, :], rhs[e] * ds
        x = np.linalg.solve(Ms, rs)
        for _ in range(3):
            r = rs.astype(np.longdouble) - Ms.astype(np.longdouble) @ x.astype(np.longdouble)
            x = x + np.linalg.solve(Ms, r.astype(np.float64))
        co = x * ds
        _check_coef(c[e], co, na)
        px, py = rng.integers(0, 1024, 2000), rng.integers(0, 1024, 2000)
        px[:4], py[:4] = [0, 0, 1023, 1023], [0, 1023, 0, 1023]
        Dref = oracle.difference_at(R, S, co, L, bid, DK, DB, px, py)
        assert np.max(np.abs(D[e][px, py] - Dref)) <= TOL_D * pb.sigma


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


def test_run_host_end_to_end(cuda_device):
    p = synth.make_pair(1)
    _, _, co, Do = _oracle_all(p.R, p.S, p.L, p.basis, p.DK, p.DB)
    plan = B.Plan(p.H, p.W, p.L, p.DK, p.DB, p.basis)
    D, c = plan.run_host(p.R, p.S)
    _check_coef(c[0], co, 3 * p.L * p.L)
    assert np.max(np.abs(D - Do)) <= TOL_D * p.sigma
    assert plan.launch_count() > 0
    plan.close()


def test_run_host_async_pipeline(cuda_device):
    """Three different pairs submitted back to back through sfft_run_host_async (two staging slots, copy streams):
    every result equals the one-call-at-a-time result of that pair."""
    import torch
    ps = [synth.make_pair(1, seed=900 + i) for i in range(3)]
    plan = B.Plan(ps[0].H, ps[0].W, ps[0].L, ps[0].DK, ps[0].DB, ps[0].basis)
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


def test_argument_and_state_errors(cuda_device):
    import torch
    for bad in [(100, 128, 7, 1, 1, 0), (128, 128, 6, 1, 1, 0), (128, 128, 7, -1, 1, 0), (128, 128, 7, 1, 1, 2),
                (64, 64, 33, 1, 1, 0), (16, 128, 3, 1, 1, 0)]:
        st, _ = B.sfft_plan_create(*bad)
        assert st == B.SFFT_ERR_INVALID_ARG, bad
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
