"""ORACLE — test infrastructure, NOT the product.

Plain, slow, FP64 NumPy implementation of the per-q polarization build written from
/root/reference/PAPER.md (arxiv 2506.03477).  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this package; the
product path (paper_2506_03477_b200) never does and shares no code with it.

What is computed (every function cites the passage it follows):

  stage (a)  z[n, n', I] = sum_{alpha,beta in site(I)} conj(C_{k+q}[alpha, n'])
                            * P_s[I, alpha, beta] * C_k[beta, n]
             -- the muffin-tin part of Eq. (8) with the eigenfunction
             expansion of Eq. (4).  z = conj(Z_paper) with
             P[I,alpha,beta] = <phi_alpha | M_I phi_beta>  (reading R1).

  weights    w_j(n, n') = -2 f_n (1 - f_n') D / (D^2 + omega_j^2),  D = eps'_{n'} - eps_n
             -- the bracket of Eq. (14) at omega = i*omega_j with
             delta -> 0 ("general complex omega where we can neglect +-i delta",
             PAPER.md:161), occupations generalised as in BASELINE.json:north_star.

  stage (b)  chi0[j][I, J] = (1/N_k) sum_k sum_{n,n' kept} w_j * conj(z_I) * z_J
             -- Eq. (14) = Alg. 1 lines 16-21 with a
             dense weight per frequency instead of histogram bins.

All parity pins live in tests/test_oracle_*.py (closed forms, brute force, invariants,
library reductions); nothing here is "parity unpinned".
"""
from __future__ import annotations

from typing import Sequence

import numpy as np


# --------------------------------------------------------------------------- weights
def pair_weights(eps_k, f_k, eps_kq, f_kq, omega, occ_tol: float = 1e-12) -> np.ndarray:
    """w[j, n, n'] of Eq. (14) on the imaginary axis.

    kept iff f_n (1 - f_n') > occ_tol (strict; reading R2); dropped pairs are exactly 0.
    D^2 + omega^2 == 0 gives 0 (reading R3: the intraband 0/0 term is dropped).
    """
    eps_k = np.asarray(eps_k, dtype=np.float64)
    eps_kq = np.asarray(eps_kq, dtype=np.float64)
    f_k = np.asarray(f_k, dtype=np.float64)
    f_kq = np.asarray(f_kq, dtype=np.float64)
    omega = np.asarray(omega, dtype=np.float64)
    D = eps_kq[None, :] - eps_k[:, None]                  # (n_o, n_u)
    occ = f_k[:, None] * (1.0 - f_kq[None, :])            # (n_o, n_u)
    den = D[None, :, :] ** 2 + omega[:, None, None] ** 2  # (n_freq, n_o, n_u)
    num = (-2.0 * occ * D)[None, :, :]
    w = np.zeros_like(den)
    np.divide(num, den, out=w, where=den != 0.0)
    w[:, ~(occ > occ_tol)] = 0.0
    return w


# --------------------------------------------------------------------------- stage (a)
def _site_offsets(sizes: Sequence[int]) -> np.ndarray:
    return np.concatenate([[0], np.cumsum(np.asarray(sizes, dtype=np.int64))])


def zmel_ref(P_sites: Sequence[np.ndarray], Ck: np.ndarray, Ckq: np.ndarray) -> np.ndarray:
    """z[n, n', I] for one k (Eq. 8 with Eq. 4), two matmul steps per site.

    P_sites[s]: (m_s, b_s, b_s) = P_s[I, alpha, beta]
    Ck:  (n_o, N_b) band-major, Ck[n, beta]  = C_k[beta, n]
    Ckq: (n_u, N_b) band-major, Ckq[n', alpha] = C_{k+q}[alpha, n']
    """
    b = [p.shape[1] for p in P_sites]
    m = [p.shape[0] for p in P_sites]
    ob, om = _site_offsets(b), _site_offsets(m)
    n_o, n_u = Ck.shape[0], Ckq.shape[0]
    z = np.zeros((n_o, n_u, int(om[-1])), dtype=np.complex128)
    for s, Ps in enumerate(P_sites):
        Cs = Ck[:, ob[s]:ob[s + 1]]                   # (n_o, b)   C_k[beta, n]
        Cqs = Ckq[:, ob[s]:ob[s + 1]]                 # (n_u, b)   C_kq[alpha, n']
        # step 1: T[I, alpha, n] = sum_beta P[I, alpha, beta] C_k[beta, n]
        T = np.matmul(Ps, Cs.T[None, :, :])           # (m, b, n_o)
        # step 2: z[n, n', I] = sum_alpha conj(C_kq[alpha, n']) T[I, alpha, n]
        Tn = np.transpose(T, (2, 1, 0))               # (n_o, b, m)
        z[:, :, om[s]:om[s + 1]] = np.matmul(np.conj(Cqs)[None, :, :], Tn)
    return z


# --------------------------------------------------------------------------- stage (b)
def chi0_accumulate_ref(acc: np.ndarray, z: np.ndarray, w: np.ndarray) -> None:
    """acc[j] += Z^H diag(w_j) Z with Z = z reshaped to (pairs, N_M)  (Eq. 14)."""
    n_m = z.shape[-1]
    Z = z.reshape(-1, n_m)
    Zh = Z.conj().T
    for j in range(w.shape[0]):
        acc[j] += Zh @ (w[j].reshape(-1, 1) * Z)


def chi0_ref(P_sites, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, omega,
             occ_tol: float = 1e-12, n_k_norm: int | None = None) -> np.ndarray:
    """chi0[j, I, J] (full matrix, NOT symmetrised) for one (q, spin).

    Ck: (n_k, n_o, N_b), Ckq: (n_k, n_u, N_b), eps/f: (n_k, n_o) and (n_k, n_u).
    Normalisation 1/N_k (reading R5); n_k_norm overrides N_k (partial sums).
    """
    n_k = Ck.shape[0]
    n_m = sum(p.shape[0] for p in P_sites)
    acc = np.zeros((len(omega), n_m, n_m), dtype=np.complex128)
    for k in range(n_k):
        z = zmel_ref(P_sites, Ck[k], Ckq[k])
        w = pair_weights(eps_k[k], f_k[k], eps_kq[k], f_kq[k], omega, occ_tol)
        chi0_accumulate_ref(acc, z, w)
    return acc / float(n_k if n_k_norm is None else n_k_norm)


def chi0_sketch_ref(P_sites, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, omega, V,
                    occ_tol: float = 1e-12, n_k_norm: int | None = None) -> np.ndarray:
    """S[j] = chi0[j] @ V without forming chi0:  sum_k Z^H (w_j o (Z V))  (exact, Eq. 14).

    Cost O(pairs * N_M * V.shape[1]); used where the full N_M^2 oracle is unaffordable.
    """
    n_k = Ck.shape[0]
    n_m = V.shape[0]
    S = np.zeros((len(omega), n_m, V.shape[1]), dtype=np.complex128)
    for k in range(n_k):
        z = zmel_ref(P_sites, Ck[k], Ckq[k])
        w = pair_weights(eps_k[k], f_k[k], eps_kq[k], f_kq[k], omega, occ_tol)
        Z = z.reshape(-1, n_m)
        ZV = Z @ V
        Zh = Z.conj().T
        for j in range(len(omega)):
            S[j] += Zh @ (w[j].reshape(-1, 1) * ZV)
    return S / float(n_k if n_k_norm is None else n_k_norm)


def chi0_entries_ref(P_sites, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, omega, rows, cols,
                     occ_tol: float = 1e-12, n_k_norm: int | None = None) -> np.ndarray:
    """Sampled entries chi0[j, rows[t], cols[t]] computed one by one (Eq. 14)."""
    rows = np.asarray(rows); cols = np.asarray(cols)
    n_k = Ck.shape[0]
    out = np.zeros((len(omega), len(rows)), dtype=np.complex128)
    for k in range(n_k):
        z = zmel_ref(P_sites, Ck[k], Ckq[k])
        w = pair_weights(eps_k[k], f_k[k], eps_kq[k], f_kq[k], omega, occ_tol)
        Z = z.reshape(-1, z.shape[-1])
        prod = np.conj(Z[:, rows]) * Z[:, cols]            # (pairs, T)
        out += w.reshape(len(omega), -1) @ prod
    return out / float(n_k if n_k_norm is None else n_k_norm)


def hermitian_finalize_ref(chi: np.ndarray) -> np.ndarray:
    """What qsgw_chi0_finalize returns: upper triangle kept, lower = conj(upper),
    Im(diag) = 0 (Hermiticity of the matrix part; reading R12)."""
    out = np.empty_like(chi)
    for j in range(chi.shape[0]):
        U = np.triu(chi[j], 1)
        d = np.real(np.diagonal(chi[j]))
        out[j] = U + U.conj().T + np.diag(d)
    return out


# --------------------------------------------------------------------------- literal loops
def chi0_ref_naive(P_sites, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, omega,
                   occ_tol: float = 1e-12) -> np.ndarray:
    """Literal pure-Python loops over (k, n, n', I, J, alpha, beta) -- tiny inputs only.

    Independent restatement of Eqs. (4), (8), (14); pins the vectorised functions.
    """
    n_k = len(Ck)
    b = [p.shape[1] for p in P_sites]
    m = [p.shape[0] for p in P_sites]
    ob, om = _site_offsets(b), _site_offsets(m)
    n_m = int(om[-1])
    n_f = len(omega)
    chi = [[[0j for _ in range(n_m)] for _ in range(n_m)] for _ in range(n_f)]
    for k in range(n_k):
        n_o, n_u = len(Ck[k]), len(Ckq[k])
        for n in range(n_o):
            for np_ in range(n_u):
                fn, fnp = float(f_k[k][n]), float(f_kq[k][np_])
                occ = fn * (1.0 - fnp)
                if not (occ > occ_tol):
                    continue
                D = float(eps_kq[k][np_]) - float(eps_k[k][n])
                zvec = [0j] * n_m
                for s in range(len(P_sites)):
                    for Il in range(m[s]):
                        acc = 0j
                        for a in range(b[s]):
                            for bt in range(b[s]):
                                acc += (complex(Ckq[k][np_][ob[s] + a]).conjugate()
                                        * complex(P_sites[s][Il][a][bt])
                                        * complex(Ck[k][n][ob[s] + bt]))
                        zvec[om[s] + Il] = acc
                for j in range(n_f):
                    om_j = float(omega[j])
                    den = D * D + om_j * om_j
                    if den == 0.0:
                        continue
                    wj = -2.0 * occ * D / den
                    for I in range(n_m):
                        zc = zvec[I].conjugate()
                        for J in range(n_m):
                            chi[j][I][J] += wj * zc * zvec[J]
    return np.array(chi, dtype=np.complex128) / float(n_k)
