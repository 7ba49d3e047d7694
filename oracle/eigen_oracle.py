"""ORACLE -- test infrastructure, NOT the product (see oracle/chi0_oracle.py for the rules).

Orthonormal mixed product basis that diagonalises the Coulomb matrix, plain NumPy/SciPy FP64, written from
/root/reference/PAPER.md section 2.3:

  |E_mu> = sum_I z_{mu I} |M_I>,   v |E_mu> = v_mu |E_mu>,   sum_J (v_IJ - v_mu O_IJ) z_{mu J} = 0,
  O_IJ = <M_I | M_J>  (Hermitian positive definite),   v_IJ = <M_I | v | M_J>  (Hermitian),
  v = sum_mu |E_mu> v_mu <E_mu|                                                                     Eq. (7)

"mu = 1 corresponds to the largest eigenvalue": eigenvalues in DESCENDING order.  {E_mu} orthonormal means
z^H O z = 1.  The result is returned as U[I, mu] = z_{mu I} (the layout qsgw_chi0_to_coulomb_basis takes: E_mu = sum_I M_I U[I, mu]).
The generalized Hermitian-definite eigenproblem is a library primitive here (scipy.linalg.eigh(v, O), LAPACK zhegvd);
eigenvectors are unique only up to a phase (and a unitary mixing inside a degenerate eigenvalue), so tests compare the
eigenvalues, the residual, the O-orthonormality and Eq. (7).  Pins: tests/test_oracle_eigen_pins.py.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg


def coulomb_eigenbasis_ref(v: np.ndarray, O: np.ndarray):
    """(v_mu descending, U[I, mu]) with v U = O U diag(v_mu), U^H O U = 1."""
    w, Z = scipy.linalg.eigh(v, O)          # ascending, Z^H O Z = 1
    order = np.argsort(-w, kind="stable")
    return w[order], Z[:, order]


def coulomb_from_eigenbasis_ref(O: np.ndarray, U: np.ndarray, v_mu: np.ndarray) -> np.ndarray:
    """Eq. (7) in the M_I representation: v_IJ = sum_mu <M_I|E_mu> v_mu <E_mu|M_J> = (O U) diag(v_mu) (O U)^H."""
    OU = O @ U
    return (OU * v_mu[None, :]) @ OU.conj().T
