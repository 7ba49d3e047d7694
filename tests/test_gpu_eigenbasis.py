"""GPU parity of the generalized eigenproblem of the Coulomb matrix in the mixed product basis (row f4; PAPER.md:116-118,
Eq. 7) through the C ABI (qsgw_coulomb_eigenbasis) against oracle.coulomb_eigenbasis_ref on the same seeded (v, O).
Eigenvectors are fixed only up to a phase (and a rotation inside a degenerate eigenvalue), so what is compared is what is
unique: the eigenvalues element by element (<= 1e-11 of the largest, FP64 on both sides, condition number of O ~ 2500), and
that the rest is valid: residual (v - v_mu O) z = 0, orthonormality z^H O z = 1, Eq. (7), and |<E_mu^oracle | E_mu^cuda>| = 1
for the non-degenerate spectrum of the generator."""
import numpy as np
import pytest

import oracle
from qsgw_synth import synthetic_mpb_matrices

pytestmark = pytest.mark.gpu


def run(v, O):
    import torch
    import paper_2506_03477_b200 as q
    vmu, U, sweeps = q.coulomb_eigenbasis(torch.from_numpy(v).cuda(), torch.from_numpy(O).cuda())
    torch.cuda.synchronize()
    return vmu.cpu().numpy(), U.cpu().numpy(), sweeps


def check(v, O, w, U, w_ref, U_ref, tol=1e-11):
    n = v.shape[0]
    assert np.all(np.diff(w) <= 0)
    assert np.abs(w - w_ref).max() <= tol * np.abs(w_ref).max()
    vn = np.linalg.norm(v)
    assert np.linalg.norm(v @ U - (O @ U) * w[None, :]) <= 1e-10 * vn
    assert np.abs(U.conj().T @ O @ U - np.eye(n)).max() <= 1e-10
    assert np.linalg.norm(oracle.coulomb_from_eigenbasis_ref(O, U, w) - v) <= 1e-10 * vn
    ov = np.abs(np.diag(U_ref.conj().T @ O @ U))
    assert np.abs(ov - 1.0).max() <= 1e-7, np.abs(ov - 1.0).max()


@pytest.mark.parametrize("n", [1, 2, 5, 63, 64, 99, 240])
def test_known_spectrum_small(n):
    v, O, lam = synthetic_mpb_matrices(n, seed=n)
    w, U, sweeps = run(v, O)
    w_ref, U_ref = oracle.coulomb_eigenbasis_ref(v, O)
    assert np.abs(w - lam).max() <= 1e-9 * lam.max()      # the spectrum the pencil was built from
    check(v, O, w, U, w_ref, U_ref)
    assert 1 <= sweeps <= 20


def test_cfg2_size():
    v, O, lam = synthetic_mpb_matrices(600, seed=6)
    w, U, sweeps = run(v, O)
    w_ref, U_ref = oracle.coulomb_eigenbasis_ref(v, O)
    check(v, O, w, U, w_ref, U_ref)


def test_only_upper_triangle_is_read_and_plane_wave_limit():
    rng = np.random.default_rng(2)
    n = 40
    kG = np.concatenate([[0.01], rng.uniform(0.5, 5.0, n - 1)])
    d = (4.0 * np.pi / kG ** 2)[rng.permutation(n)]
    v = np.diag(d).astype(np.complex128)
    O = np.eye(n, dtype=np.complex128)
    v_l = v.copy(); O_l = O.copy()
    v_l[np.tril_indices(n, -1)] = 7.0 + 3.0j               # garbage below the diagonal must not matter
    O_l[np.tril_indices(n, -1)] = -2.0 + 1.0j
    w, U, _ = run(v_l, O_l)
    assert np.allclose(w, np.sort(d)[::-1], rtol=1e-13)
    assert np.allclose(np.abs(U), np.eye(n)[:, np.argsort(-d)], atol=1e-12)


def test_not_positive_definite_overlap():
    import torch
    import paper_2506_03477_b200 as q
    v, O, _ = synthetic_mpb_matrices(70, seed=3)
    O = O.copy()
    O[5, 5] = -1.0
    with pytest.raises(q.QsgwError) as e:
        q.coulomb_eigenbasis(torch.from_numpy(v).cuda(), torch.from_numpy(O).cuda())
    assert e.value.code == 1 and "positive definite" in str(e.value)
    v2, O2, _ = synthetic_mpb_matrices(70, seed=3)                      # and the valid call still works
    w, U, _ = run(v2, O2)
    assert np.abs(w - oracle.coulomb_eigenbasis_ref(v2, O2)[0]).max() <= 1e-11 * w.max()


def test_cfg4_size():
    """N_M = 2400 (the bench size): eigenvalues against LAPACK on the same pencil, residual, orthonormality, overlaps."""
    v, O, lam = synthetic_mpb_matrices(2400, seed=1)
    w, U, sweeps = run(v, O)
    w_ref, U_ref = oracle.coulomb_eigenbasis_ref(v, O)
    assert np.abs(w - lam).max() <= 1e-9 * lam.max()
    check(v, O, w, U, w_ref, U_ref)


@pytest.mark.parametrize("n", [99, 240])
def test_elementwise_rounds_option(n):
    """Process-wide option "eig_blocked" = 0: the element-wise parallel Jacobi rounds (the first round-2 version, kept for
    comparison) give the same eigenvalues and a valid basis."""
    import paper_2506_03477_b200 as q
    v, O, lam = synthetic_mpb_matrices(n, seed=n + 1)
    w_ref, U_ref = oracle.coulomb_eigenbasis_ref(v, O)
    q.set_global_option("eig_blocked", 0)
    try:
        w0, U0, _ = run(v, O)
    finally:
        q.set_global_option("eig_blocked", 1)
    w1, U1, _ = run(v, O)
    check(v, O, w0, U0, w_ref, U_ref)
    check(v, O, w1, U1, w_ref, U_ref)
