"""ORACLE -- test infrastructure, NOT the product (see oracle/chi0_oracle.py for the rules).

Interstitial-plane-wave (IPW) block of the matrix elements, plain NumPy FP64, written from
/root/reference/PAPER.md Eqs. (4), (5) and (8).

Eq. (4): Psi_kn(r) = sum_{R u} alpha phi + sum_G beta^{kn}_G P^k_G(r);  Eq. (5): P^k_G(r) = exp(i (k + G).r) outside the
muffin tins, 0 inside.  For the product functions of the mixed product basis that are IPWs, M_I = P^{k_I}_{G_I}, the
matrix element of Eq. (8) before the rotation to E_mu is an integral over the interstitial region only (M_I vanishes
inside every MT, and outside the MTs Psi is its plane-wave part):

  <P_{G_I} Psi_{n'} | Psi_n> = sum_{alpha, beta} conj(beta^{n'}_{G_alpha}) beta^{n}_{G_beta}
                                 int_I exp(i (G_beta - G_alpha - G_I).r) d^3r            (crystal momenta: k' + k_I = k)
                             = Omega sum_{alpha, beta} conj(beta^{n'}_alpha) theta(G_beta - G_alpha - G_I) beta^{n}_beta,

  theta(G) = (1/Omega) int_cell Theta_I(r) exp(i G.r) d^3r      (Fourier coefficients of the interstitial indicator).

DESIGN.md reading R21: the paper prints no formula for this block (it cites Kotani's mixed basis, Ref. 29); the above is
what Eqs. (4), (5), (8) fix.  Convention as for the muffin-tin block (oracle.zmel_ref, R1): per unit cell volume
(the factor Omega is dropped, i.e. eigenfunctions normalised to the cell), bands n' of the conjugated side index the
SECOND band index:

  z[n, n', I] = sum_{alpha, beta} conj(Bkq[n', alpha]) Ptheta[I, alpha, beta] Bk[n, beta],
  Ptheta[I, alpha, beta] = theta(g_k[beta] - g_kq[alpha] - g_ipw[I])                 (integer reciprocal vectors),

the same bilinear form as the MT block with a structured "product tensor".  theta is an INPUT (a table on an integer box,
zero outside it).  Pins: tests/test_oracle_ipw_pins.py (a real-space quadrature that never forms theta differences, the
empty-lattice limit, the exchange symmetry, explicit loops).
"""
from __future__ import annotations

import numpy as np


def ipw_product_tensor(theta: np.ndarray, L, g_kq: np.ndarray, g_k: np.ndarray, g_ipw: np.ndarray) -> np.ndarray:
    """Ptheta[I, alpha, beta] = theta[g_k[beta] - g_kq[alpha] - g_ipw[I] + L], zero where the difference leaves the box."""
    L = np.asarray(L, dtype=np.int64)
    d = (g_k[None, None, :, :].astype(np.int64) - g_kq[None, :, None, :].astype(np.int64)
         - g_ipw[:, None, None, :].astype(np.int64)) + L                       # (I, alpha, beta, 3)
    ok = np.all((d >= 0) & (d <= 2 * L), axis=-1)
    d = np.clip(d, 0, 2 * L)
    return np.where(ok, theta[d[..., 0], d[..., 1], d[..., 2]], 0.0)


def zmel_ipw_ref(theta, L, g_kq, g_k, g_ipw, Bk: np.ndarray, Bkq: np.ndarray) -> np.ndarray:
    """z[n, n', I] of the IPW block; Bk (n_o, N_k), Bkq (n_u, N_kq).  Two matmul steps as in zmel_ref."""
    P = ipw_product_tensor(theta, L, g_kq, g_k, g_ipw)        # (I, alpha, beta)
    T = np.matmul(P, Bk.T[None, :, :])                        # (I, alpha, n)   T = sum_beta P[I, alpha, beta] Bk[n, beta]
    Tn = np.transpose(T, (2, 1, 0))                           # (n, alpha, I)
    return np.matmul(np.conj(Bkq)[None, :, :], Tn)            # (n, n', I)


def zmel_ipw_naive(theta, L, g_kq, g_k, g_ipw, Bk, Bkq) -> np.ndarray:
    """Explicit loops (tiny sizes)."""
    n_o, n_u, n_i = Bk.shape[0], Bkq.shape[0], g_ipw.shape[0]
    z = np.zeros((n_o, n_u, n_i), dtype=np.complex128)
    for i in range(n_i):
        for a in range(g_kq.shape[0]):
            for b in range(g_k.shape[0]):
                d = g_k[b].astype(int) - g_kq[a].astype(int) - g_ipw[i].astype(int)
                if np.any(np.abs(d) > np.asarray(L)):
                    continue
                th = theta[d[0] + L[0], d[1] + L[1], d[2] + L[2]]
                for n in range(n_o):
                    for m in range(n_u):
                        z[n, m, i] += np.conj(Bkq[m, a]) * th * Bk[n, b]
    return z
