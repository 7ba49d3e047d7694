"""Pins of the W^c oracle (Eqs. 10, 19) against what the mathematics fixes: the scalar
closed form, the defining identity eps eps^-1 = 1, the Neumann series, the spectral form through an independent
library routine (eigh), a Cholesky solve, sign / Hermiticity invariants, and the chi0 -> 0 limit."""
import numpy as np
import pytest
import scipy.linalg

import oracle
from qsgw_synth import coulomb_eigenvalues, generate, get_config


def _chi_and_v(idx=0, n_k=None):
    cfg = get_config(idx)
    prob = generate(cfg, n_k=n_k)
    sp = prob.spins[0]
    sites = [prob.P_site(s) for s in range(cfg.n_sites)]
    chi = oracle.hermitian_finalize_ref(oracle.chi0_ref(sites, sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                                                        prob.omega))
    return chi, coulomb_eigenvalues(cfg)


def test_scalar_closed_form():
    # N_M = 1: eps = 1 - v chi, W^c = v (1/(1 - v chi) - 1) = v^2 chi / (1 - v chi)
    chi = np.array([[[-0.37 + 0j]], [[-0.02 + 0j]]])
    v = np.array([2.5])
    w = oracle.wc_ref(chi, v)
    for j in range(2):
        c = chi[j, 0, 0].real
        assert w[j, 0, 0] == pytest.approx(2.5 ** 2 * c / (1 - 2.5 * c), rel=1e-14)
    assert oracle.dielectric_ref(chi, v)[0, 0, 0] == pytest.approx(1 + 2.5 * 0.37, rel=1e-15)


def test_defining_identity_and_invariants():
    chi, v = _chi_and_v(0)
    eps = oracle.dielectric_ref(chi, v)
    w = oracle.wc_ref(chi, v)
    sv = np.sqrt(v)
    eye = np.eye(len(v))
    for j in range(chi.shape[0]):
        inv = w[j] / sv[:, None] / sv[None, :] + eye              # eps^-1 recovered from W^c
        assert np.linalg.norm(eps[j] @ inv - eye) <= 1e-11 * np.linalg.norm(eps[j])
        assert np.linalg.norm(w[j] - w[j].conj().T) <= 1e-12 * np.linalg.norm(w[j])     # Hermitian
        # chi0(i omega) <= 0 (cfg 0: all D > 0)  =>  eps >= 1  =>  eps^-1 <= 1  =>  W^c <= 0, and eps > 0
        assert np.linalg.eigvalsh(eps[j]).min() >= 1.0 - 1e-12
        assert np.linalg.eigvalsh((w[j] + w[j].conj().T) / 2).max() <= 1e-10
    # weaker screening at larger omega: |W^c| decreases (chi0 decays monotonically, pinned in test_oracle_pins)
    nrm = np.linalg.norm(w.reshape(w.shape[0], -1), axis=1)
    assert np.all(np.diff(nrm) < 0)


def test_spectral_form_and_cholesky_route():
    chi, v = _chi_and_v(1, n_k=4)
    sv = np.sqrt(v)
    w = oracle.wc_ref(chi, v)
    for j in (0, 7, 15):
        B = -(sv[:, None] * chi[j] * sv[None, :])                 # eps = 1 + B, B Hermitian >= 0
        lam, U = np.linalg.eigh(B)
        w_spec = sv[:, None] * ((U * (1.0 / (1.0 + lam) - 1.0)) @ U.conj().T) * sv[None, :]
        assert np.linalg.norm(w[j] - w_spec) <= 1e-11 * np.linalg.norm(w_spec)
        c = scipy.linalg.cho_factor(np.eye(len(v)) + B, lower=True)
        w_chol = sv[:, None] * (scipy.linalg.cho_solve(c, np.eye(len(v))) - np.eye(len(v))) * sv[None, :]
        assert np.linalg.norm(w[j] - w_chol) <= 1e-11 * np.linalg.norm(w_chol)


def test_neumann_series_and_zero_limit():
    rng = np.random.default_rng(5)
    n = 12
    a = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    chi = -(a @ a.conj().T)[None] * 1e-6                           # small: ||sqrt(v) chi sqrt(v)|| << 1
    v = rng.uniform(0.5, 3.0, n)
    sv = np.sqrt(v)
    X = sv[:, None] * chi[0] * sv[None, :]                         # eps = 1 - X, eps^-1 - 1 = X + X^2 + X^3 + ...
    series = X + X @ X + X @ X @ X + X @ X @ X @ X
    w = oracle.wc_ref(chi, v)[0]
    assert np.linalg.norm(w - sv[:, None] * series * sv[None, :]) <= 1e-10 * np.linalg.norm(w)
    assert np.all(oracle.wc_ref(np.zeros((2, n, n), dtype=complex), v) == 0.0)


def test_coulomb_eigenvalue_recipe():
    for idx in range(5):
        cfg = get_config(idx)
        v = coulomb_eigenvalues(cfg)
        assert v.shape == (cfg.n_m,) and np.all(v > 0) and np.array_equal(v, coulomb_eigenvalues(cfg))
        assert 0.8 * 4 * np.pi / (0.3 + 0.05 * (cfg.n_m - 1)) <= v.min() and v.max() <= 1.25 * 4 * np.pi / 0.3


def test_rotation_equals_rotating_z_before_accumulation():
    """Pins the index / conjugation convention of rotate_to_coulomb_basis_ref against the definition: rotating
    the matrix elements, z_mu = sum_I U[I, mu] z_I, and accumulating gives the same chi0 as U^H chi0 U."""
    from qsgw_synth import haar_unitary
    cfg = get_config(0)
    prob = generate(cfg, n_k=2)
    sp = prob.spins[0]
    sites = [prob.P_site(s) for s in range(cfg.n_sites)]
    rng = np.random.default_rng(11)
    U = haar_unitary(rng, cfg.n_m)
    acc_I = np.zeros((len(prob.omega), cfg.n_m, cfg.n_m), dtype=np.complex128)
    acc_mu = np.zeros_like(acc_I)
    for k in range(2):
        z = oracle.zmel_ref(sites, sp.Ck[k], sp.Ckq[k])
        w = oracle.pair_weights(sp.eps_k[k], sp.f_k[k], sp.eps_kq[k], sp.f_kq[k], prob.omega)
        oracle.chi0_accumulate_ref(acc_I, z, w)
        oracle.chi0_accumulate_ref(acc_mu, z @ U, w)               # z_mu[n, n', mu] = sum_I z[n, n', I] U[I, mu]
    rot = oracle.rotate_to_coulomb_basis_ref(acc_I, U)
    assert np.linalg.norm(rot - acc_mu) <= 1e-13 * np.linalg.norm(acc_mu)
    # unitary invariants and the trivial cases
    for j in (0, 3):
        assert np.allclose(np.linalg.eigvalsh((rot[j] + rot[j].conj().T) / 2),
                           np.linalg.eigvalsh((acc_I[j] + acc_I[j].conj().T) / 2), rtol=1e-11, atol=1e-13)
        assert np.trace(rot[j]) == pytest.approx(np.trace(acc_I[j]), rel=1e-12)
    assert np.array_equal(oracle.rotate_to_coulomb_basis_ref(acc_I, np.eye(cfg.n_m)), acc_I)
    U2 = haar_unitary(rng, cfg.n_m)
    assert np.allclose(oracle.rotate_to_coulomb_basis_ref(rot, U2), oracle.rotate_to_coulomb_basis_ref(acc_I, U @ U2),
                       rtol=1e-11, atol=1e-14)
