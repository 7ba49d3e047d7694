"""ORACLE -- test infrastructure, NOT the product (see oracle/chi0_oracle.py for the rules).

Screened Coulomb interaction on the imaginary axis from the polarization, plain NumPy FP64:

  eps[j]   = 1 - sqrt(v) chi0[j] sqrt(v)                       Eq. (10)
  W^c[j]   = sqrt(v) (eps[j]^-1 - 1) sqrt(v)                   Eq. (19), PAPER.md:179-182  (Eq. 11 minus the bare v)

v_mu > 0 are the Coulomb eigenvalues of the product basis (a diagonal matrix in the paper's E_mu basis,
Eq. 10); chi0 is the Hermitian matrix produced by the chi0 build.  The inverse is numpy.linalg.inv of the
definition -- no factorisation shortcuts, so that the GPU path (Cholesky) is checked against an independent route.
Pins: tests/test_oracle_wc_pins.py.
"""
from __future__ import annotations

import numpy as np


def dielectric_ref(chi0: np.ndarray, v: np.ndarray) -> np.ndarray:
    """eps[j] = delta - sqrt(v_mu) chi0[j]_{mu nu} sqrt(v_nu)   (Eq. 10)."""
    sv = np.sqrt(np.asarray(v, dtype=np.float64))
    chi0 = np.asarray(chi0, dtype=np.complex128)
    eye = np.eye(chi0.shape[-1], dtype=np.complex128)
    return eye[None, :, :] - sv[None, :, None] * chi0 * sv[None, None, :]


def wc_ref(chi0: np.ndarray, v: np.ndarray) -> np.ndarray:
    """W^c[j] = sqrt(v) (eps[j]^-1 - 1) sqrt(v)   (Eq. 19)."""
    sv = np.sqrt(np.asarray(v, dtype=np.float64))
    eps = dielectric_ref(chi0, v)
    eye = np.eye(eps.shape[-1], dtype=np.complex128)
    out = np.empty_like(eps)
    for j in range(eps.shape[0]):
        out[j] = sv[:, None] * (np.linalg.inv(eps[j]) - eye) * sv[None, :]
    return out


def rotate_to_coulomb_basis_ref(chi0: np.ndarray, U: np.ndarray) -> np.ndarray:
    """chi0 in the orthonormal basis E_mu = sum_I M_I U[I, mu] that diagonalises the Coulomb matrix (Eq. 7,
    PAPER.md:118; Z in terms of E_mu, Eq. 8):  z_mu = sum_I U[I, mu] z_I, hence
    chi0_{mu nu} = sum_{IJ} conj(U[I, mu]) chi0_{IJ} U[J, nu] = (U^H chi0 U)_{mu nu}  for every frequency."""
    U = np.asarray(U, dtype=np.complex128)
    return np.stack([U.conj().T @ c @ U for c in np.asarray(chi0, dtype=np.complex128)])
