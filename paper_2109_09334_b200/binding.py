"""Thin ctypes binding of libsfft_b200 (include/sfft.h): argument marshalling only.

Functions carry the C names (sfft_plan_create, sfft_build_system, sfft_solve, sfft_subtract,
sfft_plan_destroy, ...).  `Plan` bundles a handle with a torch-owned workspace; torch is used
for device memory and the stream only -- every step of the path runs in the library's kernels.
There is no CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes
import os

import numpy as np

from . import build as _build

SFFT_BASIS_POLY, SFFT_BASIS_BSPLINE = 0, 1
SFFT_OK, SFFT_ERR_INVALID_ARG, SFFT_ERR_STATE, SFFT_ERR_WORKSPACE, SFFT_ERR_CUDA, SFFT_ERR_NOT_SPD = range(6)

# every symbol include/sfft.h declares (checked against the built library by tests/test_abi_and_host.py)
EXPORTS = [
    "sfft_plan_create", "sfft_plan_create_rect", "sfft_plan_set_batch", "sfft_plan_set_stream", "sfft_plan_set_const_phot_ratio", "sfft_plan_set_corr_route", "sfft_plan_num_solved", "sfft_plan_num_unknowns",
    "sfft_plan_num_kernel_terms", "sfft_plan_num_background_terms", "sfft_plan_workspace_bytes",
    "sfft_plan_set_workspace", "sfft_build_system", "sfft_get_system", "sfft_get_lag_table", "sfft_solve",
    "sfft_subtract", "sfft_mask_fill", "sfft_mask_fill_static", "sfft_static_last_error", "sfft_decorrelate", "sfft_plan_set_reuse_spectra", "sfft_plan_status", "sfft_plan_host_staging_bytes", "sfft_plan_set_host_staging",
    "sfft_run_host", "sfft_run_host_async", "sfft_run_host_wait", "sfft_run_host_f32", "sfft_run_host_async_f32", "sfft_plan_launch_count", "sfft_plan_destroy",
    "sfft_strerror", "sfft_last_cuda_error", "sfft_version", "sfft_plan_profile", "sfft_plan_profile_read",
]
SFFT_NUM_STAGES = 10
STAGE_NAMES = ["rowfft", "corr", "lagsum", "moments", "gather", "solve", "subtract_prep", "subtract", "subtract_fir",
               "subtract_inverse"]

_lib = None


class SfftError(RuntimeError):
    def __init__(self, status, where, detail=""):
        self.status = status
        msg = f"{where}: {sfft_strerror(status)}"
        super().__init__(msg + (f" [{detail}]" if detail else ""))


def library_path():
    return _build.LIB


def load_library(build_if_missing=True):
    """dlopen libsfft_b200.so (building it with nvcc first if absent).  Raises if unavailable."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_build.LIB) and not build_if_missing:
        raise FileNotFoundError(f"{_build.LIB} is missing: run __graft_entry__.build()")
    if build_if_missing:
        _build.build_library()          # no-op unless the library is missing or older than its sources
    L = ctypes.CDLL(_build.LIB)
    vp, ci, cs = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    pvp, pci = ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(ctypes.c_int)
    sig = {
        "sfft_plan_create": (ci, [pvp, ci, ci, ci, ci, ci, ci]),
        "sfft_plan_create_rect": (ci, [pvp, ci, ci, ci, ci, ci, ci, ci]),
        "sfft_plan_set_batch": (ci, [vp, ci]),
        "sfft_plan_set_stream": (ci, [vp, vp]),
        "sfft_plan_set_const_phot_ratio": (ci, [vp, ci]),
        "sfft_plan_set_corr_route": (ci, [vp, ci]),
        "sfft_plan_num_solved": (ci, [vp]),
        "sfft_plan_num_unknowns": (ci, [vp]),
        "sfft_plan_num_kernel_terms": (ci, [vp]),
        "sfft_plan_num_background_terms": (ci, [vp]),
        "sfft_plan_workspace_bytes": (cs, [vp]),
        "sfft_plan_set_workspace": (ci, [vp, vp, cs]),
        "sfft_build_system": (ci, [vp, vp, vp]),
        "sfft_get_system": (ci, [vp, pvp, pvp, pci]),
        "sfft_get_lag_table": (ci, [vp, ci, pvp, ctypes.POINTER(cs), ctypes.POINTER(cs)]),
        "sfft_solve": (ci, [vp, vp]),
        "sfft_subtract": (ci, [vp, vp, vp, vp, vp]),
        "sfft_mask_fill": (ci, [vp, vp, vp, ctypes.c_double, ctypes.c_double, ci, ci, vp, vp, vp]),
        "sfft_mask_fill_static": (ci, [vp, vp, ci, ci, ctypes.c_double, ctypes.c_double, ci, ci, vp, vp, vp, vp]),
        "sfft_static_last_error": (ctypes.c_char_p, []),
        "sfft_decorrelate": (ci, [vp, vp, vp, vp, ci, ci, vp, ci, vp, ci, vp, ci, vp]),
        "sfft_plan_set_reuse_spectra": (ci, [vp, ci]),
        "sfft_plan_status": (ci, [vp, pci]),
        "sfft_plan_host_staging_bytes": (cs, [vp]),
        "sfft_plan_set_host_staging": (ci, [vp, vp, cs]),
        "sfft_run_host": (ci, [vp, vp, vp, vp, vp]),
        "sfft_run_host_async": (ci, [vp, vp, vp, vp, vp]),
        "sfft_run_host_wait": (ci, [vp]),
        "sfft_run_host_f32": (ci, [vp, vp, vp, vp, vp]),
        "sfft_run_host_async_f32": (ci, [vp, vp, vp, vp, vp]),
        "sfft_plan_launch_count": (ctypes.c_long, [vp]),
        "sfft_plan_destroy": (None, [vp]),
        "sfft_strerror": (ctypes.c_char_p, [ci]),
        "sfft_last_cuda_error": (ctypes.c_char_p, [vp]),
        "sfft_version": (ctypes.c_char_p, []),
        "sfft_plan_profile": (ci, [vp, ci]),
        "sfft_plan_profile_read": (ci, [vp, vp, pci]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


# ---- one Python function per C entry point (same names, same argument order) ----

def sfft_strerror(status):
    return load_library().sfft_strerror(int(status)).decode()


def sfft_version():
    return load_library().sfft_version().decode()


def sfft_plan_create(H, W, L, DK, DB, basis):
    h = ctypes.c_void_p()
    st = load_library().sfft_plan_create(ctypes.byref(h), H, W, L, DK, DB, basis)
    return st, h


def sfft_plan_create_rect(H, W, L0, L1, DK, DB, basis):
    h = ctypes.c_void_p()
    st = load_library().sfft_plan_create_rect(ctypes.byref(h), H, W, L0, L1, DK, DB, basis)
    return st, h


def sfft_plan_set_batch(plan, nbatch):
    return load_library().sfft_plan_set_batch(plan, nbatch)


def sfft_plan_set_stream(plan, stream_ptr):
    return load_library().sfft_plan_set_stream(plan, ctypes.c_void_p(stream_ptr))


def sfft_plan_set_const_phot_ratio(plan, on):
    return load_library().sfft_plan_set_const_phot_ratio(plan, int(on))


def sfft_plan_set_corr_route(plan, route):
    return load_library().sfft_plan_set_corr_route(plan, int(route))


def sfft_plan_num_solved(plan):
    return load_library().sfft_plan_num_solved(plan)


def sfft_plan_num_unknowns(plan):
    return load_library().sfft_plan_num_unknowns(plan)


def sfft_plan_workspace_bytes(plan):
    return load_library().sfft_plan_workspace_bytes(plan)


def sfft_plan_set_workspace(plan, dptr, nbytes):
    return load_library().sfft_plan_set_workspace(plan, ctypes.c_void_p(dptr), nbytes)


def sfft_build_system(plan, d_R, d_S):
    return load_library().sfft_build_system(plan, ctypes.c_void_p(d_R), ctypes.c_void_p(d_S))


def sfft_get_system(plan):
    M, r, ld = ctypes.c_void_p(), ctypes.c_void_p(), ctypes.c_int()
    st = load_library().sfft_get_system(plan, ctypes.byref(M), ctypes.byref(r), ctypes.byref(ld))
    return st, M.value, r.value, ld.value


def sfft_get_lag_table(plan, which):
    t, cnt, stride = ctypes.c_void_p(), ctypes.c_size_t(), ctypes.c_size_t()
    st = load_library().sfft_get_lag_table(plan, which, ctypes.byref(t), ctypes.byref(cnt), ctypes.byref(stride))
    return st, t.value, cnt.value, stride.value


def sfft_solve(plan, d_coef):
    return load_library().sfft_solve(plan, ctypes.c_void_p(d_coef))


def sfft_subtract(plan, d_coef, d_R, d_S, d_D):
    return load_library().sfft_subtract(plan, ctypes.c_void_p(d_coef), ctypes.c_void_p(d_R), ctypes.c_void_p(d_S),
                                        ctypes.c_void_p(d_D))


def sfft_mask_fill(plan, d_R, d_S, sat_R, sat_S, rd, rb, d_Rm, d_Sm, d_mask):
    return load_library().sfft_mask_fill(plan, ctypes.c_void_p(d_R), ctypes.c_void_p(d_S), float(sat_R), float(sat_S),
                                         int(rd), int(rb), ctypes.c_void_p(d_Rm), ctypes.c_void_p(d_Sm),
                                         ctypes.c_void_p(d_mask))


SFFT_STATIC_MAX_PIXELS = 4096 * 4096


def sfft_mask_fill_static(d_R, d_S, H, W, sat_R, sat_S, rd, rb, d_Rm, d_Sm, d_mask, stream_ptr=0):
    """sfft_mask_fill for one pair without a plan or a workspace: the call allocates no device memory (its scratch is
    an array inside the library, good for H*W <= SFFT_STATIC_MAX_PIXELS).  All five images are device pointers the
    caller owns.  See include/sfft.h for who this is for and for the sharing rules."""
    return load_library().sfft_mask_fill_static(ctypes.c_void_p(d_R), ctypes.c_void_p(d_S), int(H), int(W), float(sat_R),
                                                float(sat_S), int(rd), int(rb), ctypes.c_void_p(d_Rm), ctypes.c_void_p(d_Sm),
                                                ctypes.c_void_p(d_mask), ctypes.c_void_p(stream_ptr))


def sfft_static_last_error():
    return load_library().sfft_static_last_error().decode()


def mask_fill_static(R, S, sat_R, sat_S, rd, rb, Rm, Sm, mask):
    """sfft_mask_fill_static on torch tensors, on torch's current stream.  For code that may not allocate on the
    device: the caller brings R, S (H x W float64, CUDA, contiguous) AND the outputs Rm, Sm (same, may be R, S
    themselves) and mask (uint8); nothing is created here.  Raises SfftError carrying the library's message, e.g. when
    the frame is larger than the built-in scratch."""
    import torch
    assert R.dim() == 2 and R.is_cuda and all(t.is_cuda and t.is_contiguous() and t.shape == R.shape for t in (S, Rm, Sm, mask))
    assert all(t.dtype == torch.float64 for t in (R, S, Rm, Sm)) and mask.dtype == torch.uint8
    st = sfft_mask_fill_static(R.data_ptr(), S.data_ptr(), R.shape[0], R.shape[1], sat_R, sat_S, rd, rb, Rm.data_ptr(),
                               Sm.data_ptr(), mask.data_ptr(), torch.cuda.current_stream(R.device).cuda_stream)
    if st != SFFT_OK:
        raise SfftError(st, "sfft_mask_fill_static", sfft_static_last_error())


def sfft_decorrelate(plan, d_coef, d_D, d_Ddc, tile, var_S, G, var_R, H):
    """var_S [nS], G [nS][LG][LG], var_R [nR], H [nR][LH][LH]: numpy (host) arrays."""
    vS, vR = np.ascontiguousarray(var_S, dtype=np.float64), np.ascontiguousarray(var_R, dtype=np.float64)
    Gk, Hk = np.ascontiguousarray(G, dtype=np.float64), np.ascontiguousarray(H, dtype=np.float64)
    assert Gk.ndim == 3 and Hk.ndim == 3 and Gk.shape[0] == vS.size and Hk.shape[0] == vR.size
    return load_library().sfft_decorrelate(plan, ctypes.c_void_p(d_coef), ctypes.c_void_p(d_D), ctypes.c_void_p(d_Ddc),
                                           int(tile), int(vS.size), vS.ctypes.data, int(Gk.shape[1]), Gk.ctypes.data,
                                           int(vR.size), vR.ctypes.data, int(Hk.shape[1]), Hk.ctypes.data)


def sfft_plan_set_reuse_spectra(plan, on):
    return load_library().sfft_plan_set_reuse_spectra(plan, int(on))


def sfft_plan_host_staging_bytes(plan):
    return load_library().sfft_plan_host_staging_bytes(plan)


def sfft_plan_set_host_staging(plan, dptr, nbytes):
    return load_library().sfft_plan_set_host_staging(plan, ctypes.c_void_p(dptr), nbytes)


def sfft_plan_status(plan):
    info = ctypes.c_int(-1)
    st = load_library().sfft_plan_status(plan, ctypes.byref(info))
    return st, info.value


def sfft_run_host(plan, h_R, h_S, h_D, h_coef):
    return load_library().sfft_run_host(plan, ctypes.c_void_p(h_R), ctypes.c_void_p(h_S), ctypes.c_void_p(h_D),
                                        ctypes.c_void_p(h_coef))


def sfft_run_host_async(plan, h_R, h_S, h_D, h_coef):
    return load_library().sfft_run_host_async(plan, ctypes.c_void_p(h_R), ctypes.c_void_p(h_S), ctypes.c_void_p(h_D),
                                              ctypes.c_void_p(h_coef))


def sfft_run_host_f32(plan, h_R, h_S, h_D, h_coef):
    return load_library().sfft_run_host_f32(plan, ctypes.c_void_p(h_R), ctypes.c_void_p(h_S), ctypes.c_void_p(h_D),
                                            ctypes.c_void_p(h_coef))


def sfft_run_host_async_f32(plan, h_R, h_S, h_D, h_coef):
    return load_library().sfft_run_host_async_f32(plan, ctypes.c_void_p(h_R), ctypes.c_void_p(h_S), ctypes.c_void_p(h_D),
                                                  ctypes.c_void_p(h_coef))


def sfft_run_host_wait(plan):
    return load_library().sfft_run_host_wait(plan)


def sfft_plan_launch_count(plan):
    return load_library().sfft_plan_launch_count(plan)


def sfft_plan_profile(plan, nsteps):
    return load_library().sfft_plan_profile(plan, nsteps)


def sfft_plan_profile_read(plan, nsteps):
    ms = np.zeros((nsteps, SFFT_NUM_STAGES))
    nrec = ctypes.c_int(0)
    st = load_library().sfft_plan_profile_read(plan, ms.ctypes.data, ctypes.byref(nrec))
    return st, ms[:nrec.value]


def sfft_plan_destroy(plan):
    load_library().sfft_plan_destroy(plan)


def sfft_last_cuda_error(plan):
    return load_library().sfft_last_cuda_error(plan).decode()


# ---- convenience: a plan plus its torch-owned workspace ----

def _basis_id(basis):
    if isinstance(basis, str):
        return {"poly": SFFT_BASIS_POLY, "bspline": SFFT_BASIS_BSPLINE}[basis]
    return int(basis)


class Plan:
    """sfft_plan handle + workspace tensor on the current CUDA device and stream."""

    def __init__(self, H, W, L, DK, DB, basis="poly", nbatch=1, device="cuda:0", const_phot_ratio=False,
                 reuse_spectra=False, corr_route=0):
        import torch
        if not torch.cuda.is_available():
            raise SfftError(SFFT_ERR_CUDA, "Plan", "no CUDA device: libsfft_b200 has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        if isinstance(L, (tuple, list)):          # rectangular kernel (L0 along x, L1 along y); layouts keep max(L0, L1)
            st, self.h = sfft_plan_create_rect(H, W, L[0], L[1], DK, DB, _basis_id(basis))
            L = max(L)
        else:
            st, self.h = sfft_plan_create(H, W, L, DK, DB, _basis_id(basis))
        if st != SFFT_OK:
            raise SfftError(st, "sfft_plan_create")
        self.H, self.W, self.L, self.nbatch = H, W, L, nbatch
        self._check(sfft_plan_set_batch(self.h, nbatch), "sfft_plan_set_batch")
        self._check(sfft_plan_set_const_phot_ratio(self.h, const_phot_ratio), "sfft_plan_set_const_phot_ratio")
        if corr_route:
            self._check(sfft_plan_set_corr_route(self.h, corr_route), "sfft_plan_set_corr_route")
        self.n = sfft_plan_num_unknowns(self.h)
        self.ns = sfft_plan_num_solved(self.h)
        self.ws_bytes = sfft_plan_workspace_bytes(self.h)
        self.ws = torch.empty(self.ws_bytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.ws.data_ptr() + 255) & ~255
        self.stream = torch.cuda.current_stream(self.device)
        self._check(sfft_plan_set_stream(self.h, self.stream.cuda_stream), "sfft_plan_set_stream")
        self._check(sfft_plan_set_workspace(self.h, ptr, self.ws_bytes), "sfft_plan_set_workspace")
        self._check(sfft_plan_set_reuse_spectra(self.h, reuse_spectra), "sfft_plan_set_reuse_spectra")
        self.staging = None

    def ensure_host_staging(self):
        """Allocate the staging area of the host-buffer entry points on first use."""
        if self.staging is None:
            nbytes = sfft_plan_host_staging_bytes(self.h)
            self.staging = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device=self.device)
            ptr = (self.staging.data_ptr() + 255) & ~255
            self._check(sfft_plan_set_host_staging(self.h, ptr, nbytes), "sfft_plan_set_host_staging")

    def _check(self, st, where):
        if st != SFFT_OK:
            raise SfftError(st, where, sfft_last_cuda_error(self.h) if st == SFFT_ERR_CUDA else "")

    def _img(self, t):
        torch = self.torch
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
        assert t.numel() == self.nbatch * self.H * self.W
        return t.data_ptr()

    def _ws_view(self, ptr, shape):
        """Clone of `shape` doubles at device pointer `ptr`, which lies inside the torch-owned workspace."""
        off, nbytes = ptr - self.ws.data_ptr(), int(np.prod(shape)) * 8
        assert 0 <= off and off + nbytes <= self.ws.numel()
        return self.ws[off:off + nbytes].view(self.torch.float64).reshape(shape).clone()

    def build_system(self, R, S):
        self._check(sfft_build_system(self.h, self._img(R), self._img(S)), "sfft_build_system")

    def solve(self, coef=None):
        torch = self.torch
        if coef is None:
            coef = torch.empty((self.nbatch, self.n), dtype=torch.float64, device=self.device)
        self._check(sfft_solve(self.h, coef.data_ptr()), "sfft_solve")
        return coef

    def subtract(self, coef, R, S, D=None):
        torch = self.torch
        if D is None:
            D = torch.empty_like(S)
        self._check(sfft_subtract(self.h, coef.data_ptr(), self._img(R), self._img(S), self._img(D)), "sfft_subtract")
        return D

    def mask_fill(self, R, S, sat_R, sat_S, rd, rb, inplace=False):
        """NEXT-2: masked pair (Rm, Sm) and the uint8 mask."""
        torch = self.torch
        Rm, Sm = (R, S) if inplace else (torch.empty_like(R), torch.empty_like(S))
        mask = torch.empty(R.shape, dtype=torch.uint8, device=self.device)
        self._check(sfft_mask_fill(self.h, self._img(R), self._img(S), sat_R, sat_S, rd, rb, Rm.data_ptr(), Sm.data_ptr(),
                                   mask.data_ptr()), "sfft_mask_fill")
        return Rm, Sm, mask

    def decorrelate(self, coef, D, tile, var_S, G, var_R, H, out=None):
        """NEXT-3 (App. C): D convolved tile by tile with the unit-sum decorrelation kernel of Eq. C20."""
        out = self.torch.empty_like(D) if out is None else out
        self._check(sfft_decorrelate(self.h, coef.data_ptr(), self._img(D), self._img(out), tile, var_S, G, var_R, H),
                    "sfft_decorrelate")
        return out

    def status(self, check=True):
        st, info = sfft_plan_status(self.h)
        if check and st != SFFT_OK:
            raise SfftError(st, "sfft_plan_status", f"info={info}")
        return st, info

    def system(self, batch=None):
        """Copies of (M [b][ns][ns], rhs [b][ns]) as torch tensors (parity tests); one batch entry if `batch` is given."""
        st, pM, pr, ld = sfft_get_system(self.h)
        self._check(st, "sfft_get_system")
        self.status()
        if batch is not None:
            return (self._ws_view(pM + 8 * batch * self.ns * ld, (self.ns, ld)),
                    self._ws_view(pr + 8 * batch * self.ns, (self.ns,)))
        return self._ws_view(pM, (self.nbatch, self.ns, ld)), self._ws_view(pr, (self.nbatch, self.ns))

    def lag_table(self, which, batch=0):
        st, pt, cnt, stride = sfft_get_lag_table(self.h, which)
        self._check(st, "sfft_get_lag_table")
        self.status()
        return self._ws_view(pt + 8 * stride * batch, (cnt,))

    def run_host(self, R_host, S_host):
        """End to end with host (numpy) buffers through sfft_run_host.  Returns (D, coef) numpy arrays."""
        self.ensure_host_staging()
        D = np.empty_like(R_host)
        coef = np.empty((self.nbatch, self.n))
        if R_host.dtype == np.float32:        # FP32 storage, FP64 arithmetic
            assert S_host.dtype == np.float32
            st = sfft_run_host_f32(self.h, R_host.ctypes.data, S_host.ctypes.data, D.ctypes.data, coef.ctypes.data)
            self._check(st, "sfft_run_host_f32")
            return D, coef
        st = sfft_run_host(self.h, R_host.ctypes.data, S_host.ctypes.data, D.ctypes.data, coef.ctypes.data)
        self._check(st, "sfft_run_host")
        return D, coef

    def profile(self, nsteps):
        self._check(sfft_plan_profile(self.h, nsteps), "sfft_plan_profile")

    def profile_read(self, nsteps):
        st, ms = sfft_plan_profile_read(self.h, nsteps)
        self._check(st, "sfft_plan_profile_read")
        return ms

    def launch_count(self):
        return sfft_plan_launch_count(self.h)

    def close(self):
        if getattr(self, "h", None):
            sfft_plan_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
