"""ORACLE -- test infrastructure, NOT the product (see oracle/chi0_oracle.py for the rules).

The paper's own real-axis route to the polarization, plain NumPy FP64, written from
/root/reference/PAPER.md Eqs. (15)-(18) in the order of Alg. 1 lines 9-27:

  spectral part   A[j][I, J] = (1/N_k) sum_k sum_{pairs p with w(p, j, k) != 0} w(p, j, k) conj(z[p, I]) z[p, J]
                  -- the matrix sum of Eq. (15) per histogram bin j = [edges[j], edges[j+1]) (Eq. 17), with the
                  pair lists of Alg. 1 line 14 and the gather / scale / GEMM of lines 16-21.  The prefactor pi/i
                  of Eq. (15) is NOT applied: A is the Hermitian, positive semidefinite bin-integrated spectral
                  weight, Im Pi = -pi A (reading R19).  z = conj(Z_paper) as everywhere (R1).
                  The weights w(p, j, k) are INPUTS in sparse form (the paper computes its tetrahedron weights,
                  Eq. 16, on the CPU before the loop, Alg. 1 line 8): per k-point a CSR-by-bin triple
                  (bin_ptr[n_bins+1], pair[nnz], w[nnz]) with pair = n * n_u + n'.
  Hilbert         chi0(i omega_i) = sum_j K[i, j] A[j]                                             Eq. (18)
                  From Eq. (14) with the spectral weight of a pair spread uniformly over its bin ("taking into
                  account the size of histogram bins"; the paper prints no formula -- reading R20):
                  1/(i omega - w') - 1/(i omega + w') = -2 w' / (w'^2 + omega^2), averaged over the bin,
                    K[i, j] = -log((R_j^2 + omega_i^2) / (L_j^2 + omega_i^2)) / (R_j - L_j),   [L_j, R_j) = bin j,
                  evaluated as -log1p((R_j^2 - L_j^2) / (L_j^2 + omega_i^2)) / (R_j - L_j).
                  (omega_i = 0 and L_j = 0 together would diverge: the caller's first edge must be > 0 then.)
Pins: tests/test_oracle_realaxis_pins.py.
"""
from __future__ import annotations

import numpy as np

from .chi0_oracle import zmel_ref


def imchi_accumulate_ref(acc: np.ndarray, z: np.ndarray, bin_ptr, pair, w) -> None:
    """acc[j] += Z_pair^dagger x W_Zpair for every bin j (Alg. 1 lines 13-21).

    z: (n_o, n_u, N_M); pair indices address its first two axes flattened (n * n_u + n')."""
    n_m = z.shape[-1]
    Z = z.reshape(-1, n_m)
    bin_ptr = np.asarray(bin_ptr)
    pair = np.asarray(pair)
    w = np.asarray(w, dtype=np.float64)
    for j in range(len(bin_ptr) - 1):
        lo, hi = int(bin_ptr[j]), int(bin_ptr[j + 1])
        if hi == lo:
            continue
        Zp = Z[pair[lo:hi]]                              # l.17: gather the contributing pairs
        WZ = w[lo:hi, None] * Zp                         # l.18: scale by the weight of (pair, bin)
        acc[j] += Zp.conj().T @ WZ                       # l.21: Im Pi += Z_pair^dagger x W_Zpair


def imchi_ref(P_sites, Ck, Ckq, weights, n_bins: int, n_k_norm: int | None = None) -> np.ndarray:
    """A[j, I, J] for one (q, spin): weights[k] = (bin_ptr, pair, w) of k-point k (Eq. 15 without pi/i)."""
    n_k = Ck.shape[0]
    n_m = sum(p.shape[0] for p in P_sites)
    acc = np.zeros((n_bins, n_m, n_m), dtype=np.complex128)
    for k in range(n_k):
        z = zmel_ref(P_sites, Ck[k], Ckq[k])
        imchi_accumulate_ref(acc, z, *weights[k])
    return acc / float(n_k if n_k_norm is None else n_k_norm)


def hilbert_matrix_imag(edges, omega_out) -> np.ndarray:
    """K[i, j] of Eq. (18) for targets on the imaginary axis (reading R20)."""
    edges = np.asarray(edges, dtype=np.float64)
    om = np.asarray(omega_out, dtype=np.float64)
    L, R = edges[:-1], edges[1:]
    # log(1 + x) form of the same ratio: well conditioned when the bin is narrow against omega
    x = ((R - L) * (R + L))[None, :] / (L[None, :] ** 2 + om[:, None] ** 2)
    return -np.log1p(x) / (R - L)[None, :]


def hilbert_matrix_real(edges, omega_out) -> np.ndarray:
    """K[i, j] of Eq. (18) for targets omega_i on the REAL axis (the paper's own use): the Hermitian
    part of Eq. (14), P[1/(omega - w') - 1/(omega + w')] = 2 w' / (omega^2 - w'^2), averaged over bin j (reading R20):
      K[i, j] = log|(omega_i^2 - L_j^2) / (omega_i^2 - R_j^2)| / (R_j - L_j).
    Logarithmically singular where omega_i sits on a bin edge: targets are taken inside bins (e.g. their centres)."""
    edges = np.asarray(edges, dtype=np.float64)
    om = np.asarray(omega_out, dtype=np.float64)
    L, R = edges[:-1], edges[1:]
    num = np.abs(om[:, None] ** 2 - L[None, :] ** 2)
    den = np.abs(om[:, None] ** 2 - R[None, :] ** 2)
    return (np.log(num) - np.log(den)) / (R - L)[None, :]


def hilbert_real_ref(A: np.ndarray, edges, omega_out) -> np.ndarray:
    """Re Pi(omega_i)[I, J] = sum_j K[i, j] A[j][I, J] on the real axis (Eq. 18)."""
    return np.tensordot(hilbert_matrix_real(edges, omega_out), A, axes=(1, 0))


def hilbert_imag_ref(A: np.ndarray, edges, omega_out) -> np.ndarray:
    """chi0(i omega_i)[I, J] = sum_j K[i, j] A[j][I, J]   (Eq. 18; Alg. 1 line 27)."""
    K = hilbert_matrix_imag(edges, omega_out)
    return np.tensordot(K, A, axes=(1, 0))


def imchi_naive(P_sites, Ck, Ckq, weights, n_bins: int) -> np.ndarray:
    """Literal loops over (k, bin, entry, I, J) with z from the 7-loop definition -- tiny inputs only."""
    n_k = len(Ck)
    n_m = sum(p.shape[0] for p in P_sites)
    out = [[[0j for _ in range(n_m)] for _ in range(n_m)] for _ in range(n_bins)]
    for k in range(n_k):
        z = zmel_ref(P_sites, np.asarray(Ck[k]), np.asarray(Ckq[k]))
        n_u = z.shape[1]
        bin_ptr, pair, w = weights[k]
        for j in range(n_bins):
            for e in range(int(bin_ptr[j]), int(bin_ptr[j + 1])):
                n, np_ = divmod(int(pair[e]), n_u)
                for I in range(n_m):
                    zc = complex(z[n, np_, I]).conjugate()
                    for J in range(n_m):
                        out[j][I][J] += float(w[e]) * zc * complex(z[n, np_, J])
    return np.array(out, dtype=np.complex128) / float(n_k)
