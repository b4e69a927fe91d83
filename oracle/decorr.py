"""CPU oracle for NEXT-3, noise decorrelation (App. C) -- TEST INFRASTRUCTURE ONLY.

Plain numpy, following the appendix step by step; numpy.fft serves as the DFT primitive.  Shares no code with
the CUDA path.  What the paper fixes, and the readings taken where it is silent (DESIGN g22):

  D = sum_j S_j (*) G_j - [sum_i R_i (*) H_i] (*) K                                        (C17)
  Q0^ = sqrt( sigma_D^2 / { sum_j s2_Sj |G_j^|^2 + sum_i s2_Ri |K^|^2 |H_i^|^2 } )         (C20)
  "SFFT simply normalizes the decorrelation kernel Q to have a unit kernel sum"
      => sigma_D^2 := the denominator at zero frequency, i.e. Q0^(0) = 1.
  "perform the operation by splitting the images into smaller segments": square tiles of `tile`
      pixels; in each tile the spatially varying kernel is frozen at the tile's centre pixel
      (x_c, y_c) = (a*tile + tile/2, b*tile + tile/2):  K(al,be) = sum_t k_{t,al be} T_t(x_c, y_c)  with k the pixel
      kernels of Eqs. 3-4 (k_{t,00} = a_{t,00} - sum_{others} a_{t,al be}) and T_t the weights of the fit;
      the tile is convolved circularly with Q (DFT of the tile x Q0^, inverse DFT): the derivation is for one
      convolution kernel on a periodic frame, and the paper gives no seam treatment.
  G_j, H_i (already divided by the number of co-added images) are the same for every tile.
"""
import numpy as np

from . import binding as _b


def pixel_kernels(coef, L, basis, DK):
    """k[t][al+w][be+w] from the delta-basis coefficients (Eqs. 3-4)."""
    FK = _b.num_terms(basis, DK)
    k = np.array(coef[:FK * L * L], dtype=np.float64).reshape(FK, L, L).copy()
    w = (L - 1) // 2
    for t in range(FK):
        others = k[t].sum() - k[t, w, w]
        k[t, w, w] = k[t, w, w] - others
    return k


def kernel_at(coef, L, basis, DK, H, W, xc, yc):
    """The matching kernel frozen at pixel (xc, yc): K(al,be) = sum_t k_t(al,be) f_i(xc) g_j(yc)."""
    k = pixel_kernels(coef, L, basis, DK)
    fx, gy = _b.axis_table(basis, H, DK), _b.axis_table(basis, W, DK)
    K = np.zeros((L, L))
    for t, (i, j) in enumerate(_b.terms(basis, DK)):
        K += k[t] * fx[i, xc] * gy[j, yc]
    return K


def _embed(kern, T):
    """Kernel with lag (al,be) at [al mod T][be mod T] of a T x T frame."""
    Lk = kern.shape[0]
    wk = (Lk - 1) // 2
    out = np.zeros((T, T))
    for a in range(Lk):
        for b in range(Lk):
            out[(a - wk) % T, (b - wk) % T] += kern[a, b]
    return out


def q0_hat(K, T, var_S, G, var_R, Hk):
    """Eq. C20 on the T x T frequency grid with the unit-sum normalisation."""
    Kh = np.fft.fft2(_embed(K, T))
    sS = sum(v * np.abs(np.fft.fft2(_embed(np.asarray(g, dtype=np.float64), T))) ** 2 for v, g in zip(var_S, G))
    sR = sum(v * np.abs(np.fft.fft2(_embed(np.asarray(h, dtype=np.float64), T))) ** 2 for v, h in zip(var_R, Hk))
    den = sS + np.abs(Kh) ** 2 * sR
    return np.sqrt(den[0, 0] / den), den


def decorrelate(D, coef, L, basis, DK, tile, var_S, G, var_R, Hk):
    """Decorrelated difference image, tile by tile."""
    D = np.asarray(D, dtype=np.float64)
    H, W = D.shape
    assert H % tile == 0 and W % tile == 0
    out = np.empty_like(D)
    for a in range(H // tile):
        for b in range(W // tile):
            K = kernel_at(coef, L, basis, DK, H, W, a * tile + tile // 2, b * tile + tile // 2)
            Q0, _ = q0_hat(K, tile, var_S, G, var_R, Hk)
            sl = (slice(a * tile, (a + 1) * tile), slice(b * tile, (b + 1) * tile))
            out[sl] = np.real(np.fft.ifft2(np.fft.fft2(D[sl]) * Q0))
    return out
