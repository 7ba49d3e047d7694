"""Pins of oracle/eigen_oracle.py (orthonormal product basis that diagonalises the Coulomb matrix, Eq. 7):
  1. a pencil built from a KNOWN spectrum: M = E S  =>  O = S^H S, v = S^H diag(lambda) S has generalized eigenvalues lambda;
  2. the plane-wave limit the paper quotes: O = 1, v = diag(4 pi / |k + G|^2): v_mu = the sorted diagonal, mu = 1 the largest
     ~ 4 pi / |k|^2;
  3. defining properties: residual of (v - v_mu O) z = 0, orthonormality z^H O z = 1, Eq. (7), descending order;
  4. invariance under a change of the non-orthogonal basis M -> M T (eigenvalues unchanged, U -> T^-1 U);
  5. a 2 x 2 case by hand."""
import numpy as np

import oracle
from qsgw_synth import synthetic_mpb_matrices


def test_known_spectrum():
    v, O, lam = synthetic_mpb_matrices(60, seed=1)
    w, U = oracle.coulomb_eigenbasis_ref(v, O)
    assert np.all(np.diff(w) <= 0)
    assert np.abs(w - lam).max() <= 1e-9 * lam.max()
    assert w[0] > 20 * w[1]                               # the 4 pi / |k|^2 eigenvalue stands out


def test_plane_wave_limit():
    rng = np.random.default_rng(3)
    kG = np.concatenate([[0.01], rng.uniform(0.5, 5.0, 19)])
    d = 4.0 * np.pi / kG ** 2
    perm = rng.permutation(20)
    w, U = oracle.coulomb_eigenbasis_ref(np.diag(d[perm]).astype(np.complex128), np.eye(20, dtype=np.complex128))
    assert np.allclose(w, np.sort(d)[::-1], rtol=1e-14)
    assert abs(w[0] - 4.0 * np.pi / 0.01 ** 2) <= 1e-9 * w[0]
    assert np.allclose(np.abs(U), np.eye(20)[:, np.argsort(-d[perm])], atol=1e-12)   # E_mu = one plane wave each


def test_defining_properties_and_eq7():
    v, O, _ = synthetic_mpb_matrices(45, seed=2)
    w, U = oracle.coulomb_eigenbasis_ref(v, O)
    assert np.linalg.norm(v @ U - (O @ U) * w[None, :]) <= 1e-10 * np.linalg.norm(v)
    assert np.abs(U.conj().T @ O @ U - np.eye(45)).max() <= 1e-10
    assert np.linalg.norm(oracle.coulomb_from_eigenbasis_ref(O, U, w) - v) <= 1e-10 * np.linalg.norm(v)
    # a dropped conjugate / transposed U in Eq. (7) fails:
    bad = (O @ U.conj() * w[None, :]) @ (O @ U.conj()).conj().T
    assert np.linalg.norm(bad - v) > 1e-3 * np.linalg.norm(v)


def test_basis_change_invariance():
    rng = np.random.default_rng(8)
    v, O, _ = synthetic_mpb_matrices(30, seed=4)
    T = rng.standard_normal((30, 30)) + 1j * rng.standard_normal((30, 30)) + 6 * np.eye(30)
    w, U = oracle.coulomb_eigenbasis_ref(v, O)
    w2, U2 = oracle.coulomb_eigenbasis_ref(T.conj().T @ v @ T, T.conj().T @ O @ T)
    assert np.abs(w - w2).max() <= 1e-9 * w.max()
    # same functions E_mu up to a phase: M T U2 = M U  =>  |U^H O (T U2)| = 1 on the diagonal
    ov = U.conj().T @ O @ (T @ U2)
    assert np.abs(np.abs(np.diag(ov)) - 1.0).max() <= 1e-8


def test_two_by_two_by_hand():
    """O = [[1, s], [s, 1]], v = [[a, 0], [0, b]]: det(v - x O) = (a - x)(b - x) - x^2 s^2 = 0."""
    a, b, s = 3.0, 1.0, 0.5
    O = np.array([[1.0, s], [s, 1.0]], dtype=np.complex128)
    v = np.diag([a, b]).astype(np.complex128)
    w, U = oracle.coulomb_eigenbasis_ref(v, O)
    q = 1.0 - s * s
    roots = np.sort(np.roots([q, -(a + b), a * b]).real)[::-1]
    assert np.allclose(w, roots, rtol=1e-13)
