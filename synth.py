"""Seeded synthetic star-field pairs for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the CPU oracle, and therefore
holds none of the method's arithmetic (no weights, no normal system, no FFT): it only
renders images.  The paper's survey images (ZTF, AST3-II, TESS, DECam 2046x4094, TMTS;
PAPER.md:232-234, 393, 756-795) are not available offline; these inputs take their
shapes, kernel widths (15-25 px) and crowded/sparse character from them.
Recipe: DESIGN.md "Input recipe" (follows SURVEY.md section 8(d)).

numpy only; deterministic for a given (config, subfield): Generator(PCG64(seed)) with
seed = 210909334 + config index (config 5 sub-field e: 210909334 + 1000 + e).
"""
from dataclasses import dataclass

import numpy as np

SEED0 = 210909334
SKY = 100.0          # ADU, both epochs
READ_SIGMA = 5.0     # ADU
SIGMA_BKG = float(np.sqrt(SKY + READ_SIGMA ** 2))  # background noise sigma, gain 1 (DESIGN g16)
STAMP_HW = 12

# H, W, L, DK, DB, basis, stars, psf, fwhm (lo, hi), transients, batch
CONFIGS = {
    1: dict(H=128, W=128, L=7, DK=1, DB=1, basis="poly", stars=60, psf="gauss", fwhm=(2.5, 2.5), transients=0, batch=1),
    2: dict(H=1024, W=1024, L=11, DK=2, DB=2, basis="poly", stars=2000, psf="moffat", fwhm=(3.0, 3.0), transients=20, batch=1),
    3: dict(H=2048, W=4096, L=15, DK=2, DB=2, basis="poly", stars=15000, psf="moffat", fwhm=(2.5, 4.0), transients=50, batch=1),
    4: dict(H=4096, W=4096, L=17, DK=2, DB=2, basis="poly", stars=40000, psf="moffat", fwhm=(3.0, 3.0), transients=0, batch=1),
    5: dict(H=1024, W=1024, L=11, DK=4, DB=4, basis="bspline", stars=2000, psf="moffat", fwhm=(3.0, 3.0), transients=20, batch=64),
}


@dataclass
class Pair:
    R: np.ndarray        # [H][W] float64 (or [B][H][W])
    S: np.ndarray
    H: int
    W: int
    L: int
    DK: int
    DB: int
    basis: str           # "poly" | "bspline"
    sigma: float         # background noise sigma used by the D tolerance
    config: int


def _coords(H, W, x0=0, x1=None):
    x1 = H if x1 is None else x1
    ux = ((2.0 * np.arange(x0, x1) + 1.0) / H - 1.0)[:, None]
    uy = ((2.0 * np.arange(W) + 1.0) / W - 1.0)[None, :]
    return ux, uy


def _render_sources(H, W, xs, ys, flux, fwhm, psf):
    """Sum of unit-integral PSFs * flux on a wrapped grid (consistent with circular convolution)."""
    n = len(xs)
    img = np.zeros(H * W)
    if n == 0:
        return img.reshape(H, W)
    off = np.arange(-STAMP_HW, STAMP_HW + 1)
    chunk = 4096
    for s in range(0, n, chunk):
        x, y, f, fw = xs[s:s + chunk], ys[s:s + chunk], flux[s:s + chunk], fwhm[s:s + chunk]
        ix, iy = np.floor(x).astype(np.int64), np.floor(y).astype(np.int64)
        gx = ix[:, None] + off[None, :]
        gy = iy[:, None] + off[None, :]
        dx = (gx - x[:, None])[:, :, None]
        dy = (gy - y[:, None])[:, None, :]
        r2 = dx * dx + dy * dy
        if psf == "gauss":
            sig = (fw / 2.3548200450309493)[:, None, None]
            prof = np.exp(-0.5 * r2 / (sig * sig))
        else:  # Moffat beta = 3
            beta = 3.0
            alpha = (fw / (2.0 * np.sqrt(2.0 ** (1.0 / beta) - 1.0)))[:, None, None]
            prof = (1.0 + r2 / (alpha * alpha)) ** (-beta)
        prof /= prof.sum(axis=(1, 2), keepdims=True)
        vals = prof * f[:, None, None]
        idx = (np.mod(gx, H)[:, :, None] * W + np.mod(gy, W)[:, None, :]).ravel()
        img += np.bincount(idx, weights=vals.ravel(), minlength=H * W)
    return img.reshape(H, W)


def _kernel_fields(cfg_index, ux, uy):
    """Per-pixel matching-kernel parameters: sigma_x, sigma_y, shift_x, shift_y (broadcastable)."""
    one = np.ones(np.broadcast_shapes(ux.shape, uy.shape))
    if cfg_index == 1:
        return 1.2 * one, 1.2 * one, 0.0 * one, 0.0 * one
    if cfg_index in (2, 5):
        sig = 1.0 + 0.5 * (ux + 1.0) * one           # 1.0 -> 2.0 linear in x
        q = 1.0 - 0.15 * (uy + 1.0) * one            # axis ratio 1.0 -> 0.7 linear in y
        return sig, sig * q, 0.0 * one, 0.0 * one
    if cfg_index == 3:
        sig = 1.0 + 0.4 * (ux * ux + uy * uy) * one  # 1.0 -> 1.8 quadratic
        return sig, sig, 0.0 * one, 0.0 * one
    sig = 1.3 + 0.25 * (ux * ux + uy * uy) + 0.15 * ux * uy   # config 4: width + centroid shift quadratic
    return sig * one, sig * one, 0.5 * ux * uy * one, 0.5 * (ux * ux - uy * uy) * one


def _scale_bkg(cfg_index, ux, uy):
    if cfg_index == 1:
        return 1.1 + 0.0 * ux * uy, 5.0 + 4.0 * ux - 3.0 * uy
    scale = 1.0 + 0.1 * (ux * ux + uy * uy - 1.0)     # in [0.9, 1.1], quadratic
    bkg = 10.0 * (0.5 * ux - 0.3 * uy + 0.4 * ux * uy + 0.3 * ux * ux - 0.2 * uy * uy)
    return scale, bkg


def _varying_blur(clean, cfg_index, L):
    """sum_{u,v} K_{x,y}(u,v) clean(x-u, y-v), kernel evaluated at the OUTPUT pixel (true Eq. 1),
    truncated to LxL, unit sum, wrap-around.  All kernels used are axis-separable Gaussians."""
    H, W = clean.shape
    w = (L - 1) // 2
    pad = np.pad(clean, w, mode="wrap")
    out = np.empty_like(clean)
    offs = np.arange(-w, w + 1, dtype=np.float64)
    rows = max(8, min(H, (1 << 21) // W))
    tmp = np.empty((rows, W))
    for x0 in range(0, H, rows):
        x1 = min(H, x0 + rows)
        ux, uy = _coords(H, W, x0, x1)
        sx, sy, dx, dy = _kernel_fields(cfg_index, ux, uy)
        gx = np.exp(-0.5 * ((offs[:, None, None] - dx[None]) / sx[None]) ** 2)
        gy = np.exp(-0.5 * ((offs[:, None, None] - dy[None]) / sy[None]) ** 2)
        gx /= gx.sum(axis=0, keepdims=True)
        gy /= gy.sum(axis=0, keepdims=True)
        acc = np.zeros((x1 - x0, W))
        inner = np.empty((x1 - x0, W))
        t = tmp[: x1 - x0]
        for iu in range(L):
            u = iu - w
            inner[:] = 0.0
            for iv in range(L):
                v = iv - w
                np.multiply(gy[iv], pad[x0 - u + w: x1 - u + w, w - v: w - v + W], out=t)
                inner += t
            np.multiply(gx[iu], inner, out=t)
            acc += t
        out[x0:x1] = acc
    return out


def make_pair(config, subfield=None, H=None, W=None, stars=None, seed=None, noise=True):
    """One (R, S) pair of config `config` (1..5).  H/W/stars override the size for scaled-down
    test cases (star and transient counts scale with area unless `stars` is given)."""
    c = dict(CONFIGS[config])
    H0, W0 = c["H"], c["W"]
    H = H0 if H is None else H
    W = W0 if W is None else W
    area = (H * W) / float(H0 * W0)
    nstars = int(round(c["stars"] * area)) if stars is None else stars
    ntrans = int(round(c["transients"] * area))
    if seed is None:
        seed = SEED0 + config if config != 5 else SEED0 + 1000 + (0 if subfield is None else subfield)
    rng = np.random.Generator(np.random.PCG64(seed))
    L = c["L"]

    xs = rng.uniform(0.0, H, nstars)
    ys = rng.uniform(0.0, W, nstars)
    # dN/dF ~ F^-1.5 on [1e2, 1e5] by inverse CDF
    a, b, g = 1e2, 1e5, -1.5
    uq = rng.uniform(0.0, 1.0, nstars)
    flux = (a ** (g + 1) + uq * (b ** (g + 1) - a ** (g + 1))) ** (1.0 / (g + 1))
    f0, f1 = c["fwhm"]
    fwhm = f0 + (f1 - f0) * (xs / H)            # varies linearly across the field when f1 != f0
    clean_R = _render_sources(H, W, xs, ys, flux, fwhm, c["psf"])

    ux, uy = _coords(H, W)
    scale, bkg = _scale_bkg(config, ux, uy)
    clean_S = scale * _varying_blur(clean_R, config, L) + bkg
    if ntrans > 0:
        m = 2 * L
        tx = rng.uniform(m, H - m, ntrans)
        ty = rng.uniform(m, W - m, ntrans)
        tf = np.exp(rng.uniform(np.log(1e3), np.log(3e4), ntrans))
        tfw = np.sqrt((f0 + (f1 - f0) * (tx / H)) ** 2 + (2.3548 * 1.5) ** 2)   # science-epoch width
        clean_S = clean_S + _render_sources(H, W, tx, ty, tf, tfw, c["psf"])
    if noise:
        R = rng.poisson(clean_R + SKY).astype(np.float64) + rng.normal(0.0, READ_SIGMA, (H, W))
        S = rng.poisson(np.maximum(clean_S + SKY, 0.0)).astype(np.float64) + rng.normal(0.0, READ_SIGMA, (H, W))
    else:
        R, S = clean_R + SKY, clean_S + SKY
    return Pair(R=R, S=S, H=H, W=W, L=L, DK=c["DK"], DB=c["DB"], basis=c["basis"], sigma=SIGMA_BKG, config=config)


_WORKER = """
import sys, numpy as np
sys.path.insert(0, {root!r})
import synth
config, lo, hi, H, W, stars, out = {args!r}
ps = [synth.make_pair(config, subfield=e, H=H, W=W, stars=stars) for e in range(lo, hi)]
np.save(out + "_R.npy", np.stack([p.R for p in ps])); np.save(out + "_S.npy", np.stack([p.S for p in ps]))
"""


def make_batch(config=5, nbatch=None, H=None, W=None, stars=None, first=0, workers=0):
    """Config 5: stack of independent sub-field pairs first .. first+nbatch-1, images [B][H][W].
    workers > 1 renders slices of the batch in that many child interpreters (identical arrays: every
    sub-field has its own seed); used by the full-size batch-of-64 test and bench only."""
    nb = CONFIGS[config]["batch"] if nbatch is None else nbatch
    if workers > 1 and nb > 1:
        import os
        import subprocess
        import sys
        import tempfile
        root = os.path.dirname(os.path.abspath(__file__))
        nw = min(workers, nb)
        cuts = [first + (nb * q) // nw for q in range(nw + 1)]
        with tempfile.TemporaryDirectory() as tmp:
            procs = []
            for q in range(nw):
                args = (config, cuts[q], cuts[q + 1], H, W, stars, os.path.join(tmp, f"part{q}"))
                procs.append(subprocess.Popen([sys.executable, "-c", _WORKER.format(root=root, args=args)]))
            for pr in procs:
                if pr.wait() != 0:
                    raise RuntimeError("synth.make_batch: a rendering child failed")
            R = np.concatenate([np.load(os.path.join(tmp, f"part{q}_R.npy")) for q in range(nw)])
            S = np.concatenate([np.load(os.path.join(tmp, f"part{q}_S.npy")) for q in range(nw)])
        c = CONFIGS[config]
        return Pair(R=R, S=S, H=R.shape[1], W=R.shape[2], L=c["L"], DK=c["DK"], DB=c["DB"], basis=c["basis"],
                    sigma=SIGMA_BKG, config=config)
    pairs = [make_pair(config, subfield=first + e, H=H, W=W, stars=stars) for e in range(nb)]
    p0 = pairs[0]
    return Pair(R=np.stack([p.R for p in pairs]), S=np.stack([p.S for p in pairs]), H=p0.H, W=p0.W, L=p0.L,
                DK=p0.DK, DB=p0.DB, basis=p0.basis, sigma=p0.sigma, config=config)
