"""Pins of oracle/realaxis_oracle.py (the paper's real-axis route: binned spectral part, Eqs. 15-17, and the Hilbert
transform, Eq. 18; Alg. 1 lines 9-27) against what the paper and the mathematics fix:

  A (Eq. 15)   literal loops on tiny inputs; sum rule sum_j A_j = (1/N_k) sum_pairs (sum_j w) conj(z) z through one
               ZGEMM; Hermitian and positive semidefinite for positive weights ("the products ... are the positive
               definite matrix"); one pair in one bin -> w |z|^2; permutation of the entries of a bin
  K (Eq. 18)   numerical quadrature of -2 w'/(w'^2 + omega^2) over the bin; narrow-bin limit = the weight of
               Eq. (14) on the imaginary axis
  chain        with every pair's weight in the single bin that holds its excitation energy, sum_j K_ij A_j converges
               to the exact imaginary-axis chi0 of Eq. (14) (oracle.chi0_ref, itself pinned) as the bins narrow,
               at first order in the bin width (a pair sits anywhere in its bin) -- the Kramers-Kronig consistency the paper states
               (PAPER.md:177).
"""
import numpy as np
import pytest
from scipy import integrate

import oracle
from oracle.realaxis_oracle import (hilbert_imag_ref, hilbert_matrix_imag, hilbert_matrix_real, hilbert_real_ref,
                                    imchi_accumulate_ref, imchi_naive, imchi_ref)
from qsgw_synth import binned_pair_weights, generate, get_config, log_bin_edges, scaled_config


def small_problem(n_k=2, seed_offset=0):
    cfg = scaled_config(get_config(0), n_k=n_k, orb_per_site=(3, 4), pb_per_site=(3, 2), n_o=2, n_u=3)
    return generate(cfg, seed_offset=seed_offset)


def sites_of(prob):
    return [prob.P_site(s) for s in range(prob.cfg.n_sites)]


def weights_of(prob, edges, rel_width=0.05):
    sp = prob.spins[0]
    return [binned_pair_weights(sp.eps_k[k], sp.f_k[k], sp.eps_kq[k], sp.f_kq[k], edges, rel_width)
            for k in range(sp.Ck.shape[0])]


def test_bruteforce_tiny():
    prob = small_problem()
    sp = prob.spins[0]
    edges = log_bin_edges(7, 0.01, 2.0)
    wts = weights_of(prob, edges, rel_width=0.3)
    assert max(len(w[1]) for w in wts) > 6              # pairs really spread over several bins
    ref = imchi_naive(sites_of(prob), sp.Ck, sp.Ckq, wts, 7)
    got = imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, 7)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


def test_sum_rule_through_one_zgemm_and_positivity():
    prob = generate(scaled_config(get_config(0), n_k=3))
    sp = prob.spins[0]
    edges = log_bin_edges(40, 0.01, 2.0)
    wts = weights_of(prob, edges)
    A = imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, 40)
    tot = np.zeros_like(A[0])
    for k in range(3):
        z = oracle.zmel_ref(sites_of(prob), sp.Ck[k], sp.Ckq[k]).reshape(-1, prob.cfg.n_m)
        wsum = np.zeros(z.shape[0])
        np.add.at(wsum, wts[k][1], wts[k][2])
        assert np.allclose(wsum, 1.0)                    # insulator, window inside the mesh: all of f (1 - f') lands
        tot += z.conj().T @ (wsum[:, None] * z)
    assert np.abs(A.sum(axis=0) - tot / 3).max() <= 1e-13 * np.abs(tot).max()
    for j in range(40):
        assert np.abs(A[j] - A[j].conj().T).max() <= 1e-14 * max(np.abs(A[j]).max(), 1e-300)
        assert np.linalg.eigvalsh(A[j]).min() >= -1e-13 * max(np.abs(A[j]).max(), 1e-300)


def test_single_entry_and_order_inside_a_bin():
    rng = np.random.default_rng(3)
    z = rng.standard_normal((2, 3, 4)) + 1j * rng.standard_normal((2, 3, 4))
    acc = np.zeros((3, 4, 4), dtype=np.complex128)
    imchi_accumulate_ref(acc, z, [0, 0, 1, 1], [4], [0.7])          # pair 4 = (n 1, n' 1) in bin 1 only
    assert np.all(acc[0] == 0) and np.all(acc[2] == 0)
    assert np.allclose(acc[1], 0.7 * np.outer(z[1, 1].conj(), z[1, 1]), rtol=1e-15)
    a1 = np.zeros_like(acc); a2 = np.zeros_like(acc)
    imchi_accumulate_ref(a1, z, [0, 3, 3, 5], [0, 2, 5, 1, 3], [0.1, 0.2, 0.3, 0.4, 0.5])
    imchi_accumulate_ref(a2, z, [0, 3, 3, 5], [5, 0, 2, 3, 1], [0.3, 0.1, 0.2, 0.5, 0.4])
    assert np.allclose(a1, a2, rtol=1e-14, atol=1e-16)


def test_hilbert_matrix_against_quadrature_and_narrow_bin_limit():
    edges = log_bin_edges(9, 0.02, 3.0)
    om = np.array([0.0, 0.05, 0.7, 20.0])
    K = hilbert_matrix_imag(edges, om)
    for i, w in enumerate(om):
        for j in range(9):
            L, R = edges[j], edges[j + 1]
            val = integrate.quad(lambda x: -2.0 * x / (x * x + w * w), L, R, epsabs=1e-14, epsrel=1e-13)[0] / (R - L)
            assert abs(K[i, j] - val) <= 1e-11 * abs(val)
    # narrow bin around D: K -> the bracket of Eq. (14) at omega = i w, 1/(iw - D) - 1/(iw + D)
    D = 0.37
    Kn = hilbert_matrix_imag([D * (1 - 1e-6), D * (1 + 1e-6)], om)
    exact = (1.0 / (1j * om - D) - 1.0 / (1j * om + D)).real
    assert np.allclose(Kn[:, 0], exact, rtol=1e-9)


def test_chain_converges_to_the_imaginary_axis_chi0():
    prob = generate(scaled_config(get_config(0), n_k=2))
    sp = prob.spins[0]
    sites = sites_of(prob)
    exact = oracle.chi0_ref(sites, sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq, prob.omega)
    errs = []
    for n_bins in (50, 200, 800):
        edges = log_bin_edges(n_bins, 0.01, 2.0)
        wts = weights_of(prob, edges, rel_width=1e-9)     # the whole weight of a pair in the bin that holds D
        A = imchi_ref(sites, sp.Ck, sp.Ckq, wts, n_bins)
        got = hilbert_imag_ref(A, edges, prob.omega)
        errs.append(max(np.linalg.norm(got[i] - exact[i]) / np.linalg.norm(exact[i]) for i in range(len(prob.omega))))
    assert errs[0] < 2e-2 and errs[2] < 2e-3
    assert errs[1] < errs[0] / 3 and errs[2] < errs[1] / 3          # 4x narrower bins -> ~4x closer (first order)
    # the sign and the normalisation: negative semidefinite at omega = 0, like Eq. (14)
    assert np.linalg.eigvalsh(0.5 * (got[0] + got[0].conj().T)).max() <= 1e-12


def test_generator_weights_are_a_partition_of_each_pair():
    """qsgw_synth.binned_pair_weights: every kept pair's entries add up to f (1 - f') and sit in bins its window
    overlaps (input recipe)."""
    prob = generate(scaled_config(get_config(2), n_k=1))
    sp = prob.spins[0]
    edges = log_bin_edges(60, 1e-3, 1.5)
    bp, pr, w = binned_pair_weights(sp.eps_k[0], sp.f_k[0], sp.eps_kq[0], sp.f_kq[0], edges, 0.05)
    assert bp[0] == 0 and bp[-1] == len(pr) == len(w) and np.all(np.diff(bp) >= 0) and np.all(w > 0)
    n_u = prob.cfg.n_u
    tot = np.zeros(prob.cfg.n_o * n_u)
    np.add.at(tot, pr, w)
    occ = (sp.f_k[0][:, None] * (1 - sp.f_kq[0][None, :])).reshape(-1)
    D = (sp.eps_kq[0][None, :] - sp.eps_k[0][:, None]).reshape(-1)
    inside = (D * 0.95 >= edges[0]) & (D * 1.05 < edges[-1]) & (occ > 1e-12)
    assert np.allclose(tot[inside], occ[inside], rtol=1e-12)
    assert np.all(tot[(D <= 0) | (occ <= 1e-12)] == 0)


def test_hilbert_matrix_real_axis_principal_value_and_limits():
    """Real-axis targets (Eq. 18 as the paper uses it): K against the Cauchy principal value computed by scipy
    (weight='cauchy') for targets inside bins, against plain quadrature for targets outside the bin, the narrow-bin
    limit 2 D / (omega^2 - D^2) = Re of the bracket of Eq. (14), and the static limit omega -> 0 shared with the
    imaginary-axis matrix."""
    edges = log_bin_edges(9, 0.02, 3.0)
    om = np.concatenate([[1e-9], 0.5 * (edges[:-1] + edges[1:])[::2], [7.0]])
    K = hilbert_matrix_real(edges, om)
    f = lambda x, w: 2.0 * x / (w * w - x * x)
    for i, w in enumerate(om):
        for j in range(9):
            L, R = edges[j], edges[j + 1]
            if L < w < R:      # 2x/(w^2 - x^2) = -[2x/(w + x)] / (x - w): Cauchy weight 1/(x - w)
                val = integrate.quad(lambda x: -2.0 * x / (w + x), L, R, weight="cauchy", wvar=w)[0] / (R - L)
            else:
                val = integrate.quad(f, L, R, args=(w,), epsabs=1e-13, epsrel=1e-12)[0] / (R - L)
            assert abs(K[i, j] - val) <= 1e-9 * max(1.0, abs(val)), (i, j, K[i, j], val)
    D = 0.37
    w = np.array([0.1, 0.3, 0.5, 2.0])
    Kn = hilbert_matrix_real([D * (1 - 1e-7), D * (1 + 1e-7)], w)
    assert np.allclose(Kn[:, 0], (1.0 / (w - D) - 1.0 / (w + D)), rtol=1e-6)
    assert np.allclose(hilbert_matrix_real(edges, [1e-9]), hilbert_matrix_imag(edges, [0.0]), rtol=1e-9)
    A = np.random.default_rng(0).standard_normal((9, 3, 3)) + 0j
    assert np.allclose(hilbert_real_ref(A, edges, om), np.einsum("ij,jab->iab", K, A))
