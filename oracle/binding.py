"""ctypes marshalling for oracle/sfft_oracle.c (TEST INFRASTRUCTURE ONLY; see __init__.py).

No arithmetic of the method lives here: every function forwards to the C routine of the
same name.  ``normal_bruteforce`` (Tier A) and ``normal_from_lags`` (Tier B) are two-call
conveniences.
"""
import ctypes
import os
import subprocess

import numpy as np

POLY, BSPLINE = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sfft_oracle.c")
_LIB = os.path.join(_HERE, "libsfft_oracle.so")
_lib = None

_D = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_I = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_ci = ctypes.c_int


def build_library(force=False):
    """Compile sfft_oracle.c -> libsfft_oracle.so with gcc (no -march=native: the .so travels)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-mavx2", "-mfma", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build_library()
    L = ctypes.CDLL(_LIB)
    L.orc_num_axis.argtypes = [_ci, _ci]
    L.orc_num_terms.argtypes = [_ci, _ci]
    L.orc_terms.argtypes = [_ci, _ci, _I, _I]
    L.orc_axis_table.argtypes = [_ci, _ci, _ci, _D]
    L.orc_num_unknowns.argtypes = [_ci] * 4
    L.orc_design_matrix.argtypes = [_ci] * 6 + [_D, _D]
    L.orc_gram.argtypes = [_ci, ctypes.c_long, _D, _D, _D, _D]
    L.orc_lag_tables.argtypes = [_ci] * 6 + [_D] * 10
    L.orc_diag_and_rhs.argtypes = [_ci] * 6 + [_D] * 4
    L.orc_gather.argtypes = [_ci] * 3 + [_D] * 10
    L.orc_solve.argtypes = [_ci, _D, _D, _D, _ci]
    L.orc_difference.argtypes = [_ci] * 6 + [_D] * 4
    L.orc_difference_at.argtypes = [_ci] * 6 + [_D] * 3 + [_ci, _I, _I, _D]
    L.orc_corr_diff_one.argtypes = [_ci, _ci, _D, _D, _ci, _ci, ctypes.POINTER(ctypes.c_double)]
    L.orc_corr_diff_one.restype = ctypes.c_double
    L.orc_weighted_ref.argtypes = [_ci] * 5 + [_D, _D]
    L.orc_num_threads.restype = _ci
    L.orc_mask_fill.argtypes = [_ci, _ci, _D, _D, ctypes.c_double, ctypes.c_double, _ci, _ci, _D, _D,
                                np.ctypeslib.ndpointer(dtype=np.uint8, flags="C_CONTIGUOUS")]
    L.orc_mask_fill.restype = ctypes.c_long
    L.orc_cpr_num_unknowns.argtypes = [_ci] * 4
    L.orc_cpr_constrain.argtypes = [_ci] * 4 + [_D] * 4
    L.orc_cpr_expand.argtypes = [_ci] * 4 + [_D] * 2
    _lib = L
    return L


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return _load().orc_num_threads()


def num_terms(basis, D):
    return _load().orc_num_terms(basis, D)


def num_axis(basis, D):
    return _load().orc_num_axis(basis, D)


def terms(basis, D):
    F = num_terms(basis, D)
    ti, tj = np.zeros(F, np.int32), np.zeros(F, np.int32)
    _load().orc_terms(basis, D, ti, tj)
    return list(zip(ti.tolist(), tj.tolist()))


def axis_table(basis, N, D):
    out = np.zeros((num_axis(basis, D), N))
    _load().orc_axis_table(basis, N, D, out)
    return out


def num_unknowns(L, basis, DK, DB):
    return _load().orc_num_unknowns(L, basis, DK, DB)


def design_matrix(R, L, basis, DK, DB):
    """Tier A: Phi as [n][P] (row k = image of unknown k, flattened)."""
    R = _c(R)
    H, W = R.shape
    n = num_unknowns(L, basis, DK, DB)
    Phi = np.zeros((n, H * W))
    _load().orc_design_matrix(H, W, L, basis, DK, DB, R, Phi)
    return Phi


def gram(Phi, S):
    Phi, S = _c(Phi), _c(S).ravel()
    n, P = Phi.shape
    M, rhs = np.zeros((n, n)), np.zeros(n)
    _load().orc_gram(n, P, Phi, S, M, rhs)
    return M, rhs


def normal_bruteforce(R, S, L, basis, DK, DB):
    """Tier A normal system from the materialised design matrix."""
    return gram(design_matrix(R, L, basis, DK, DB), S)


def diag_and_rhs(R, S, L, basis, DK, DB):
    """(diag(M), rhs) from the column definitions, without the rest of the normal matrix."""
    R, S = _c(R), _c(S)
    H, W = R.shape
    n = num_unknowns(L, basis, DK, DB)
    diag, rhs = np.zeros(n), np.zeros(n)
    _load().orc_diag_and_rhs(H, W, L, basis, DK, DB, R, S, diag, rhs)
    return diag, rhs


def lag_tables(R, S, L, basis, DK, DB):
    """Tier B: direct-sum lag tables (dict of arrays; layout in sfft_oracle.c)."""
    R, S = _c(R), _c(S)
    H, W = R.shape
    FK, FB, nO = num_terms(basis, DK), num_terms(basis, DB), 2 * L - 1
    t = dict(
        Qom=np.zeros((FK, FK, nO, nO)), Om0=np.zeros((FK, FK)),
        Qla=np.zeros((FK, FB, L, L)), La0=np.zeros((FK, FB)),
        Qth=np.zeros((FK, L, L)), Th0=np.zeros(FK),
        Phi0=np.zeros((FB, FB)), De0=np.zeros(FB),
    )
    _load().orc_lag_tables(H, W, L, basis, DK, DB, R, S, t["Qom"], t["Om0"], t["Qla"], t["La0"],
                           t["Qth"], t["Th0"], t["Phi0"], t["De0"])
    return t


def gather(t, L):
    FK, FB = t["Om0"].shape[0], t["De0"].shape[0]
    n = FK * L * L + FB
    M, rhs = np.zeros((n, n)), np.zeros(n)
    _load().orc_gather(L, FK, FB, t["Qom"], t["Om0"], t["Qla"], t["La0"], t["Qth"], t["Th0"],
                       t["Phi0"], t["De0"], M, rhs)
    return M, rhs


def normal_from_lags(R, S, L, basis, DK, DB):
    """Tier B normal system."""
    return gather(lag_tables(R, S, L, basis, DK, DB), L)


def solve(M, rhs, refine=2):
    M, rhs = _c(M), _c(rhs)
    n = rhs.shape[0]
    c = np.zeros(n)
    info = _load().orc_solve(n, M, rhs, c, refine)
    if info != 0:
        raise np.linalg.LinAlgError(f"oracle: matrix not SPD at pivot {info - 1}")
    return c


def difference(R, S, c, L, basis, DK, DB):
    R, S, c = _c(R), _c(S), _c(c)
    H, W = R.shape
    D = np.zeros((H, W))
    _load().orc_difference(H, W, L, basis, DK, DB, R, S, c, D)
    return D


def difference_at(R, S, c, L, basis, DK, DB, px, py):
    R, S, c = _c(R), _c(S), _c(c)
    H, W = R.shape
    px = np.ascontiguousarray(px, np.int32)
    py = np.ascontiguousarray(py, np.int32)
    out = np.zeros(px.shape[0])
    _load().orc_difference_at(H, W, L, basis, DK, DB, R, S, c, px.shape[0], px, py, out)
    return out


def corr_diff_one(A, B, rho, eps):
    """(q, c0) with q = sum A(x)[B(x+lag) - B(x)], c0 = sum A B, for one lag."""
    A, B = _c(A), _c(B)
    H, W = A.shape
    c0 = ctypes.c_double(0.0)
    q = _load().orc_corr_diff_one(H, W, A, B, rho, eps, ctypes.byref(c0))
    return q, c0.value


def weighted_ref(R, basis, DK, t):
    R = _c(R)
    H, W = R.shape
    out = np.zeros((H, W))
    _load().orc_weighted_ref(H, W, basis, DK, t, R, out)
    return out


def cpr_num_unknowns(L, basis, DK, DB):
    """NEXT-1 (constant photometric ratio): number of unknowns n' = n - (F_K - 1)."""
    return _load().orc_cpr_num_unknowns(L, basis, DK, DB)


def cpr_constrain(M, rhs, L, basis, DK, DB):
    """M' = C^T M C, rhs' = C^T rhs of the constant-kernel-integral model."""
    M, rhs = _c(M), _c(rhs)
    nr = cpr_num_unknowns(L, basis, DK, DB)
    Mc, rc = np.zeros((nr, nr)), np.zeros(nr)
    _load().orc_cpr_constrain(L, basis, DK, DB, M, rhs, Mc, rc)
    return Mc, rc


def cpr_expand(cr, L, basis, DK, DB):
    """c = C c' (full coefficient layout, constrained entries filled in)."""
    cr = _c(cr)
    c = np.zeros(num_unknowns(L, basis, DK, DB))
    _load().orc_cpr_expand(L, basis, DK, DB, cr, c)
    return c


def rect_select(L0, L1, basis, DK, DB):
    """NEXT-4, rectangular kernels (the delta basis spans L0 x L1 pixels).  Indices, in the layout of the
    enclosing square L = max(L0, L1), of the unknowns of the L0 x L1 model: kernel unknowns with |alpha| <= (L0-1)/2
    and |beta| <= (L1-1)/2, then the background unknowns.  The rectangular model is the square one without the other
    basis images, so its normal system is the sub-matrix M[sel][:, sel], rhs[sel] (no arithmetic involved)."""
    L = max(L0, L1)
    w, w0, w1 = (L - 1) // 2, (L0 - 1) // 2, (L1 - 1) // 2
    FK, FB = num_terms(basis, DK), num_terms(basis, DB)
    sel = [t * L * L + (al + w) * L + (be + w) for t in range(FK) for al in range(-w0, w0 + 1) for be in range(-w1, w1 + 1)]
    sel += [FK * L * L + s for s in range(FB)]
    return np.array(sel, dtype=np.int64)


def rect_expand(cs, L0, L1, basis, DK, DB):
    """Coefficients of the L0 x L1 model in the layout of the enclosing square (zeros outside the rectangle)."""
    c = np.zeros(num_unknowns(max(L0, L1), basis, DK, DB))
    c[rect_select(L0, L1, basis, DK, DB)] = cs
    return c


def mask_fill(R, S, sat_R, sat_S, rd, rb):
    """NEXT-2 (DESIGN g21): joint saturation mask grown by rd, masked pixels replaced by the mean of the
    unmasked pixels in the (2 rb + 1)^2 neighbourhood.  Returns (Rm, Sm, mask uint8)."""
    R, S = _c(R), _c(S)
    H, W = R.shape
    Rm, Sm, mask = np.zeros((H, W)), np.zeros((H, W)), np.zeros((H, W), np.uint8)
    _load().orc_mask_fill(H, W, R, S, float(sat_R), float(sat_S), int(rd), int(rb), Rm, Sm, mask)
    return Rm, Sm, mask
