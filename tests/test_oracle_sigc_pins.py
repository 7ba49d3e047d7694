"""Pins of oracle/sigc_oracle.py (imaginary-axis correlation self-energy I^c, Eqs. 22-23, PAPER.md:197-205;
Alg. 2 lines 12-25, 44) against what the paper and the mathematics fix -- none of them
re-types the oracle's formulas:

  weights   numerical quadrature (scipy.integrate.quad) of K(dE, omega) hat_i(omega); partition of unity
            sum_i w_i = atan(omega_max / dE) / pi -> sign(dE)/2 (Eq. 23 with X = 1); exactness for piecewise-linear
            X; oddness in dE; the complex two-sided form of Eq. (23) int d omega / 2 pi X / (dE - i omega)
  scalar    N_M = 1, W^c(i omega) = a / (omega^2 + b^2): closed form by residues  a sign(dE) / (2 b (|dE| + b))
  I^c       literal loops of Eq. (22) on tiny inputs; degenerate eps_q -> Hermitian and <= 0 for W^c <= 0 ... ;
            linearity in W^c; gauge invariance; a single ZGEMM per frequency through numpy.matmul.
"""
import numpy as np
import pytest
from scipy import integrate

import oracle
from oracle.sigc_oracle import imag_axis_weights, sigc_imag_naive, sigc_imag_ref, sigc_zw_ref


def mesh(n=12, w1=0.01, wmax=20.0):
    return np.concatenate([[0.0], np.geomspace(w1, wmax, n - 1)])


def K(dE, w):
    return dE / (dE * dE + w * w) / np.pi


def test_weights_match_numerical_quadrature_of_the_hat_functions():
    om = mesh(9)
    for dE in (-0.7, -0.03, 0.004, 0.2, 3.0):
        w = imag_axis_weights(np.float64(dE), om)
        for i in range(len(om)):
            val = 0.0
            if i > 0:
                a, b = om[i - 1], om[i]
                val += integrate.quad(lambda x: K(dE, x) * (x - a) / (b - a), a, b, epsabs=1e-14, epsrel=1e-13)[0]
            if i < len(om) - 1:
                a, b = om[i], om[i + 1]
                val += integrate.quad(lambda x: K(dE, x) * (b - x) / (b - a), a, b, epsabs=1e-14, epsrel=1e-13)[0]
            assert abs(w[i] - val) <= 1e-11 * max(1.0, abs(val)), (dE, i, w[i], val)


def test_weights_partition_of_unity_and_eq23_limit():
    """X = 1: sum_i w_i = int_0^{omega_max} K = atan(omega_max/dE)/pi, which tends to sign(dE)/2, the value of
    int d omega / 2 pi 1 / (dE - i omega) (Eq. 23)."""
    om = mesh(16)
    dE = np.array([-1.3, -0.2, -1e-3, 1e-3, 0.05, 0.9])
    w = imag_axis_weights(dE, om)
    assert np.allclose(w.sum(axis=0), np.arctan(om[-1] / dE) / np.pi, rtol=0, atol=1e-14)
    far = mesh(16, wmax=1e9)
    assert np.allclose(imag_axis_weights(dE, far).sum(axis=0), 0.5 * np.sign(dE), atol=2e-9)


def test_weights_odd_in_dE_zero_at_zero_and_real():
    om = mesh(10)
    dE = np.array([0.0, 0.3, -0.3, 1e-8, -1e-8])
    w = imag_axis_weights(dE, om)
    assert w.dtype == np.float64
    assert np.all(w[:, 0] == 0.0)
    assert np.allclose(w[:, 1], -w[:, 2], rtol=0, atol=1e-16)
    assert np.allclose(w[:, 3], -w[:, 4], rtol=0, atol=1e-16)
    # dE -> 0+: all the weight goes to omega_0 = 0 (K tends to delta(omega)/2)
    assert abs(w[0, 3] - 0.5) < 1e-5 and np.abs(w[1:, 3]).max() < 1e-5


def test_weights_exact_for_piecewise_linear_X_against_complex_two_sided_integral():
    """Eq. (23) as printed: int_{-inf}^{inf} d omega / 2 pi X(i omega) / (dE - i omega) with an even, piecewise-linear
    X that vanishes beyond omega_max -- evaluated by quad on the COMPLEX integrand over both half axes."""
    om = mesh(8, w1=0.05, wmax=6.0)
    rng = np.random.default_rng(5)
    xv = rng.uniform(0.2, 1.0, len(om))
    xv[-1] = 0.0                                   # continuous at omega_max: X = 0 beyond
    X = lambda w_: np.interp(abs(w_), om, xv, right=0.0)
    for dE in (-0.4, 0.15, 1.1):
        re = integrate.quad(lambda x: (X(x) / (dE - 1j * x)).real, -om[-1], om[-1], points=list(om[1:-1]) + list(-om[1:-1]) + [0.0],
                            epsabs=1e-13, epsrel=1e-12, limit=400)[0] / (2 * np.pi)
        im = integrate.quad(lambda x: (X(x) / (dE - 1j * x)).imag, -om[-1], om[-1], points=list(om[1:-1]) + list(-om[1:-1]) + [0.0],
                            epsabs=1e-13, epsrel=1e-12, limit=400)[0] / (2 * np.pi)
        got = float(imag_axis_weights(np.float64(dE), om) @ xv)
        assert abs(im) < 1e-10
        assert abs(got - re) <= 1e-10, (dE, got, re)


def test_scalar_lorentzian_closed_form_by_residues():
    """N_M = 1, one k, one intermediate state, z = 1, W^c(i omega) = a/(omega^2 + b^2):
    I^c = -a sign(dE) / (2 b (|dE| + b)) up to the quadrature error of a fine, far-reaching mesh."""
    a, b = -0.8, 0.6
    om = np.concatenate([[0.0], np.geomspace(1e-4, 1e5, 4000)])
    wc = (a / (om ** 2 + b ** 2)).reshape(-1, 1, 1).astype(np.complex128)
    z = np.ones((1, 1, 1), dtype=np.complex128)
    for e_q, e_qk in ((0.3, -0.2), (-0.25, 0.4), (0.05, 0.049)):
        dE = e_q - e_qk
        got = sigc_imag_ref([z], np.array([e_q]), [np.array([e_qk])], [wc], om)[0, 0]
        exact = -a * np.sign(dE) / (2.0 * b * (abs(dE) + b))
        assert abs(got.imag) < 1e-15
        assert abs(got.real - exact) <= 2e-6 * abs(exact), (dE, got, exact)


def tiny_case(seed, n_k=2, n_all=3, n_qp=2, n_m=3, n_f=4):
    rng = np.random.default_rng(seed)
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    om = mesh(n_f, w1=0.1, wmax=5.0)
    z = [c(n_all, n_qp, n_m) for _ in range(n_k)]
    eps_q = rng.uniform(-0.5, 0.5, n_qp)
    eps_qk = [rng.uniform(-0.6, 1.0, n_all) for _ in range(n_k)]
    wc = []
    for _ in range(n_k):
        g = c(n_f, n_m, n_m)
        wc.append(-(g @ np.conj(np.transpose(g, (0, 2, 1)))) / (1.0 + om[:, None, None] ** 2))   # Hermitian, <= 0
    return z, eps_q, eps_qk, wc, om


@pytest.mark.parametrize("seed", [0, 1])
def test_bruteforce_tiny(seed):
    z, eps_q, eps_qk, wc, om = tiny_case(seed)
    ref = sigc_imag_naive(z, eps_q, eps_qk, wc, om)
    got = sigc_imag_ref(z, eps_q, eps_qk, wc, om)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


def test_non_hermitian_w_and_transposed_operand_are_caught():
    """W^c of Eq. (22) enters as W[mu, nu] with mu on the conjugated Z: a NON-Hermitian test matrix tells
    W from W^T and W^H; the brute-force loops are the reference."""
    z, eps_q, eps_qk, wc, om = tiny_case(3)
    rng = np.random.default_rng(9)
    wc = [w + 0.5 * (rng.standard_normal(w.shape) + 1j * rng.standard_normal(w.shape)) for w in wc]
    ref = sigc_imag_naive(z, eps_q, eps_qk, wc, om)
    got = sigc_imag_ref(z, eps_q, eps_qk, wc, om)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    wrong = sigc_imag_ref(z, eps_q, eps_qk, [np.transpose(w, (0, 2, 1)) for w in wc], om)
    assert np.abs(wrong - ref).max() > 1e-3 * np.abs(ref).max()


def test_one_zgemm_per_frequency_library_reduction():
    """For one k: I^c = -sum_i (diag-scaled Z) W_i Z^H summed over n' -- through plain numpy.matmul per (i, n')."""
    z, eps_q, eps_qk, wc, om = tiny_case(4, n_k=1, n_all=4, n_qp=3, n_m=5, n_f=6)
    got = sigc_imag_ref(z, eps_q, eps_qk, wc, om)
    acc = np.zeros((3, 3), dtype=np.complex128)
    for a in range(4):
        for i in range(len(om)):
            w = imag_axis_weights(eps_q - eps_qk[0][a], om)[i]            # (n_qp,)
            acc -= np.diag(w) @ z[0][a] @ wc[0][i] @ z[0][a].conj().T
    assert np.abs(got - acc).max() <= 1e-13 * np.abs(acc).max()


def test_degenerate_eps_q_gives_hermitian_and_definite_sign():
    """Equal eps_qn for all n: the weight no longer depends on the row index, so with Hermitian W^c the matrix
    I^c is Hermitian; with all dE > 0 (weights > 0) and W^c <= 0 it is -(sum of w Z W Z^H) >= 0."""
    z, _, eps_qk, wc, om = tiny_case(6, n_k=2, n_all=4, n_qp=3, n_m=4, n_f=5)
    eps_q = np.full(3, 2.0)                         # above every eps_qk: dE > 0
    got = sigc_imag_ref(z, eps_q, eps_qk, wc, om)
    assert np.abs(got - got.conj().T).max() <= 1e-13 * np.abs(got).max()
    assert np.linalg.eigvalsh(0.5 * (got + got.conj().T)).min() >= -1e-13
    got2 = sigc_imag_ref(z, np.full(3, -3.0), eps_qk, wc, om)     # dE < 0: opposite sign
    assert np.linalg.eigvalsh(0.5 * (got2 + got2.conj().T)).max() <= 1e-13


def test_linearity_gauge_and_normalisation():
    z, eps_q, eps_qk, wc, om = tiny_case(7)
    base = sigc_imag_ref(z, eps_q, eps_qk, wc, om)
    # linear in W^c
    twice = sigc_imag_ref(z, eps_q, eps_qk, [2.5 * w for w in wc], om)
    assert np.allclose(twice, 2.5 * base, rtol=1e-13, atol=0)
    # phase of an intermediate state n' drops out; phases of the q states n rotate I^c as D I^c D^H
    rng = np.random.default_rng(1)
    ph_a = np.exp(1j * rng.uniform(0, 6.28, z[0].shape[0]))
    ph_n = np.exp(1j * rng.uniform(0, 6.28, z[0].shape[1]))
    z2 = [zz * ph_a[:, None, None] * ph_n[None, :, None] for zz in z]
    rot = sigc_imag_ref(z2, eps_q, eps_qk, wc, om)
    assert np.allclose(rot, ph_n[:, None] * base * np.conj(ph_n)[None, :], rtol=1e-12, atol=1e-15)
    # 1/N_k: a partial sum normalised by the full N_k adds up
    part = sum(sigc_imag_ref([z[k]], eps_q, [eps_qk[k]], [wc[k]], om, n_k_norm=len(z)) for k in range(len(z)))
    assert np.allclose(part, base, rtol=1e-13, atol=1e-16)


def test_zw_shape_and_chain_with_zmel_and_wc_oracles():
    """End-to-end chain of the oracles on a small cell: z from zmel_ref (Ck = C_{q-k}, Ckq = C_q), W^c from wc_ref of
    chi0_ref -- I^c finite, and ZW^c has the (n', n, nu) layout of Alg. 2 l.12."""
    from qsgw_synth import coulomb_eigenvalues, generate, get_config, scaled_config
    cfg = scaled_config(get_config(0), n_k=2)
    prob = generate(cfg)
    sp = prob.spins[0]
    sites = [prob.P_site(s) for s in range(cfg.n_sites)]
    chi = oracle.hermitian_finalize_ref(oracle.chi0_ref(sites, sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq, prob.omega))
    wc = oracle.wc_ref(chi, coulomb_eigenvalues(cfg))
    z = oracle.zmel_ref(sites, sp.Ckq[0], sp.Ck[0])          # n' over the 28 "all" states, n over 8 q states
    zw = sigc_zw_ref(z, sp.eps_k[0], sp.eps_kq[0], wc, prob.omega)
    assert zw.shape == (cfg.n_u, cfg.n_o, cfg.n_m)
    ic = sigc_imag_ref([z], sp.eps_k[0], [sp.eps_kq[0]], [wc], prob.omega)
    assert ic.shape == (cfg.n_o, cfg.n_o) and np.isfinite(ic).all() and np.abs(ic).max() > 0
