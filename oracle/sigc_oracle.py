"""ORACLE -- test infrastructure, NOT the product (see oracle/chi0_oracle.py for the rules).

Imaginary-axis part I^c of the correlation self-energy, plain NumPy FP64, written from
/root/reference/PAPER.md Eqs. (22)-(23) in the order of Alg. 2 lines 12-25 and 44
(PAPER.md:438-462,499):

  I^c_nm(q, eps_qn) = - sum_{k,n'} sum_i w^I_i(eps_qn - eps_{q-k,n'})
                        sum_{mu,nu} [Z_mu^{q-k n', q n}]^* W^c_{mu nu}(k, i omega_i) Z_nu^{q-k n', q m}      Eq. (22)

with z = conj(Z_paper) (reading R1): z[n', n, mu] is what oracle.zmel_ref returns for
Ck = C_{q-k} (rows n', the n_all intermediate states) and Ckq = C_q (rows n, the n_qp states), so
[Z_mu^{n' n}]^* = z[n', n, mu] and Z_nu^{n' m} = conj(z[n', m, nu]).

Alg. 2 per k-point and band batch:
  l.18  Z_w(mu, n', n) = Z(mu, n', n) w^I_i(eps_qn - eps_{q-k n'})
  l.23  ZW^c(n', n, nu) += sum_mu Z_w^dagger(n' n, mu) W^c_i(mu, nu)          (GEMM, repeated over omega_i)
  l.44  Sigma^c(n, m)   += sum_{n', nu} ZW^c(nu, n', n) Z(nu, n', m)          (GEMM)
The sign of Eq. (22) and the 1/N_k of reading R5 are applied once at the end (reading R18).

Weights w^I (Eq. 23).  The paper defers to Aryasetiawan-Gunnarsson and prints no formula.
DESIGN.md reading R17: with X(i omega) = X(-i omega) ("W^c(omega) = W^c(-omega)")
  int_{-inf}^{inf} d omega / 2 pi  X(i omega) / (dE - i omega) = int_0^inf d omega  K(dE, omega) X(i omega),
  K(dE, omega) = (1/pi) dE / (dE^2 + omega^2),
and the weights integrate K EXACTLY against the piecewise-linear interpolant of X on the mesh
0 = omega_0 < omega_1 < ... < omega_{n-1}, X = 0 beyond the last point:
  w_i(dE) = int hat_i(omega) K(dE, omega) d omega     (hat_i = the mesh's hat function at omega_i).
dE = 0 gives w = 0 (the principal value of an odd integrand).  The weights are real.
Pins: tests/test_oracle_sigc_pins.py.
"""
from __future__ import annotations

import numpy as np


def imag_axis_weights(dE, omega) -> np.ndarray:
    """w[i, ...] = w^I(dE, i omega_i) of Eq. (23) (reading R17), for an array dE of any shape.

    Per mesh interval [a, b] (h = b - a), with the antiderivatives
      I0 = int_a^b K = (atan(b/dE) - atan(a/dE)) / pi
      I1 = int_a^b omega K = dE / (2 pi) * log((dE^2 + b^2) / (dE^2 + a^2))
    the two hat halves contribute  (b I0 - I1)/h  to the left node and  (I1 - a I0)/h  to the right node.
    """
    omega = np.asarray(omega, dtype=np.float64)
    dE = np.asarray(dE, dtype=np.float64)
    n = omega.shape[0]
    w = np.zeros((n,) + dE.shape, dtype=np.float64)
    nz = dE != 0.0
    d = np.where(nz, dE, 1.0)
    for i in range(n - 1):
        a, b = omega[i], omega[i + 1]
        h = b - a
        I0 = (np.arctan(b / d) - np.arctan(a / d)) / np.pi
        I1 = d / (2.0 * np.pi) * np.log((d * d + b * b) / (d * d + a * a))
        w[i] += np.where(nz, (b * I0 - I1) / h, 0.0)
        w[i + 1] += np.where(nz, (I1 - a * I0) / h, 0.0)
    return w


def sigc_zw_ref(z: np.ndarray, eps_q, eps_qk, wc: np.ndarray, omega) -> np.ndarray:
    """ZW^c[n', n, nu] of Alg. 2 lines 15-25 for one k-point.

    z:  (n_all, n_qp, N_M)  z[n', n, mu] = conj(Z_mu^{q-k n', q n})
    eps_q: (n_qp,) energies eps_qn;  eps_qk: (n_all,) energies eps_{q-k, n'}
    wc: (n_freq, N_M, N_M)  W^c(k, i omega_i);  omega: (n_freq,) the mesh, omega_0 = 0
    """
    n_all, n_qp, n_m = z.shape
    dE = np.asarray(eps_q, dtype=np.float64)[None, :] - np.asarray(eps_qk, dtype=np.float64)[:, None]   # (n', n)
    w = imag_axis_weights(dE, omega)                                                                   # (i, n', n)
    zw = np.zeros((n_all * n_qp, n_m), dtype=np.complex128)
    Z = z.reshape(n_all * n_qp, n_m)
    for i in range(len(omega)):
        Zw = w[i].reshape(-1, 1) * Z                 # l.18: the weight-scaled operand
        zw += Zw @ wc[i]                             # l.23: ZW^c += Z_w^dagger x W^c
    return zw.reshape(n_all, n_qp, n_m)


def sigc_imag_ref(z_list, eps_q, eps_qk_list, wc_list, omega, n_k_norm: int | None = None) -> np.ndarray:
    """I^c[n, m] of Eq. (22) for one q: sum over the k-points given (z_list[k], eps_qk_list[k], wc_list[k]).

    Normalisation 1/N_k (reading R18, as R5 for chi0); n_k_norm overrides N_k (partial sums).
    NOT Hermitian in (n, m): the weight carries eps_qn of the row index only (Eq. 3 symmetrises later).
    """
    n_qp = z_list[0].shape[1]
    acc = np.zeros((n_qp, n_qp), dtype=np.complex128)
    for z, e_qk, wc in zip(z_list, eps_qk_list, wc_list):
        zw = sigc_zw_ref(z, eps_q, e_qk, wc, omega)
        # l.44: Sigma^c(n, m) += sum_{n', nu} ZW^c(n', n, nu) Z_paper(nu, n', m),  Z_paper = conj(z)
        acc += np.einsum("anv,amv->nm", zw, np.conj(z))
    return -acc / float(len(z_list) if n_k_norm is None else n_k_norm)


def sigc_imag_naive(z_list, eps_q, eps_qk_list, wc_list, omega) -> np.ndarray:
    """Literal loops over (k, n', n, m, i, mu, nu) of Eq. (22) -- tiny inputs only; the weight of every term
    is evaluated on its own through imag_axis_weights (scalar dE)."""
    n_qp = z_list[0].shape[1]
    out = [[0j for _ in range(n_qp)] for _ in range(n_qp)]
    for z, e_qk, wc in zip(z_list, eps_qk_list, wc_list):
        n_all, _, n_m = z.shape
        for a in range(n_all):
            for n in range(n_qp):
                w = imag_axis_weights(np.float64(eps_q[n] - e_qk[a]), omega)
                for m in range(n_qp):
                    s = 0j
                    for i in range(len(omega)):
                        for mu in range(n_m):
                            for nu in range(n_m):
                                s += w[i] * z[a, n, mu] * wc[i][mu, nu] * np.conj(z[a, m, nu])
                    out[n][m] -= s
    return np.array(out, dtype=np.complex128) / float(len(z_list))
