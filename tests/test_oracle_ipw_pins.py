"""Pins of oracle/ipw_oracle.py (IPW block of the matrix elements, Eqs. 4, 5, 8) against things
other than itself:
  1. a real-space quadrature on a periodic grid that multiplies the sampled functions point by point (no reciprocal-space
     differences, no theta look-ups): exact for band-limited functions when theta is the DFT of the sampled indicator;
  2. the empty lattice (no muffin tins): theta = delta, z = sum over the plane waves with g_beta = g_alpha + g_I;
  3. exchange symmetry conj(z[n, n', I]) = z'[n', n, -I] of the roles of the two eigenfunctions (theta(-g) = conj theta(g));
  4. explicit loops;
  5. the generator's closed-form theta: theta(0) = interstitial volume fraction, Hermitian, and convergence of the DFT of
     a sampled indicator towards it.
"""
import numpy as np

import oracle
from qsgw_synth import synthetic_ipw
from qsgw_synth.ipw import interstitial_theta


def small_lists(rng, n_kq=5, n_k=6, n_i=4, span=2):
    def pick(n):
        g = set()
        while len(g) < n:
            g.add(tuple(int(x) for x in rng.integers(-span, span + 1, 3)))
        return np.array(sorted(g), dtype=np.int32)
    return pick(n_kq), pick(n_k), pick(n_i)


def theta_box_from_mask(mask, L):
    """theta(g) = (1/N^3) sum_r mask(r) exp(+2 pi i g.r / N) for every integer g in [-L, L] (periodic in N)."""
    N = mask.shape[0]
    dft = np.fft.ifftn(mask)                      # (1/N^3) sum mask exp(+2 pi i g r / N)
    ax = [np.arange(-l, l + 1) % N for l in L]
    return dft[np.ix_(*ax)]


def test_real_space_quadrature_identity():
    rng = np.random.default_rng(11)
    N = 9
    mask = (rng.random((N, N, N)) < 0.6).astype(np.float64)     # any indicator: the identity is algebraic
    g_kq, g_k, g_i = small_lists(rng)
    L = np.array([6, 6, 6])
    theta = theta_box_from_mask(mask, L)
    n_o, n_u = 3, 4
    Bk = rng.standard_normal((n_o, len(g_k))) + 1j * rng.standard_normal((n_o, len(g_k)))
    Bkq = rng.standard_normal((n_u, len(g_kq))) + 1j * rng.standard_normal((n_u, len(g_kq)))
    r = np.stack(np.meshgrid(*([np.arange(N)] * 3), indexing="ij"), axis=-1).reshape(-1, 3)

    def waves(g):                                                # (n_g, N^3): exp(2 pi i g.r / N)
        return np.exp(2j * np.pi * (g.astype(np.float64) @ r.T) / N)
    psi = Bk @ waves(g_k)                                        # Psi_n(r), plane-wave part
    psiq = Bkq @ waves(g_kq)                                     # Psi_n'(r)
    pw_i = waves(g_i)                                            # P_{G_I}(r) / indicator
    m = mask.reshape(-1)
    z_real = np.einsum("r,ir,mr,nr->nmi", m, np.conj(pw_i), np.conj(psiq), psi) / N ** 3
    z = oracle.zmel_ipw_ref(theta, L, g_kq, g_k, g_i, Bk, Bkq)
    assert np.abs(z - z_real).max() <= 1e-13 * np.abs(z_real).max()
    # a transposed operand, a dropped conjugate or a wrong sign of g_I fail this:
    z_bad = oracle.zmel_ipw_ref(theta, L, g_kq, g_k, -g_i, Bk, Bkq)
    assert np.abs(z_bad - z_real).max() > 1e-3 * np.abs(z_real).max()
    z_bad = oracle.zmel_ipw_ref(np.conj(theta), L, g_kq, g_k, g_i, Bk, Bkq)
    assert np.abs(z_bad - z_real).max() > 1e-3 * np.abs(z_real).max()


def test_empty_lattice_limit():
    rng = np.random.default_rng(5)
    g_kq, g_k, g_i = small_lists(rng, 7, 9, 6)
    L = np.array([6, 6, 6])
    theta = np.zeros((13, 13, 13), dtype=np.complex128)
    theta[6, 6, 6] = 1.0
    Bk = rng.standard_normal((2, len(g_k))) + 1j * rng.standard_normal((2, len(g_k)))
    Bkq = rng.standard_normal((3, len(g_kq))) + 1j * rng.standard_normal((3, len(g_kq)))
    where = {tuple(g): b for b, g in enumerate(g_k)}
    ref = np.zeros((2, 3, len(g_i)), dtype=np.complex128)
    for i, gi in enumerate(g_i):
        for a, ga in enumerate(g_kq):
            b = where.get(tuple(ga + gi))
            if b is not None:
                ref[:, :, i] += Bk[:, b][:, None] * np.conj(Bkq[:, a])[None, :]
    z = oracle.zmel_ipw_ref(theta, L, g_kq, g_k, g_i, Bk, Bkq)
    assert np.abs(ref).max() > 0
    assert np.abs(z - ref).max() <= 1e-14 * np.abs(ref).max()


def test_exchange_symmetry_and_loops():
    p = synthetic_ipw(n_o=3, n_u=4, cut_pw=1.2, cut_ipw=1.5, a0=6.5, seed=3)
    z = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    zs = oracle.zmel_ipw_ref(p.theta, p.L, p.g_k, p.g_kq, -p.g_ipw, p.Bkq, p.Bk)     # roles exchanged, IPW -G_I
    assert np.abs(np.conj(z) - np.transpose(zs, (1, 0, 2))).max() <= 1e-14 * np.abs(z).max()
    zn = oracle.zmel_ipw_naive(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    assert np.abs(z - zn).max() <= 1e-14 * np.abs(z).max()
    # differences outside the box contribute zero (documented behaviour of the boundary)
    Ls = np.maximum(p.L - 1, 0)
    sl = tuple(slice(int(a - b), int(a + b) + 1) for a, b in zip(p.L, Ls))
    z_small = oracle.zmel_ipw_ref(p.theta[sl], Ls, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    zn_small = oracle.zmel_ipw_naive(p.theta[sl], Ls, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    assert np.abs(z_small - zn_small).max() <= 1e-14 * np.abs(z).max()


def test_generator_theta_closed_form():
    p = synthetic_ipw(a0=7.0, n_spheres=2, seed=1)
    c = tuple(int(l) for l in p.L)
    vol = abs(np.linalg.det(p.A))
    assert abs(p.theta[c] - (1.0 - np.sum(4.0 * np.pi * p.radii ** 3 / 3.0) / vol)) <= 1e-14
    assert np.abs(p.theta[::-1, ::-1, ::-1] - np.conj(p.theta)).max() <= 1e-15
    # DFT of the sampled indicator -> the closed form as the grid refines (indicator: first-order convergence)
    errs = []
    L = np.array([2, 2, 2])
    th = interstitial_theta(p.A, p.tau, p.radii, L)
    for N in (24, 48):
        f = (np.stack(np.meshgrid(*([np.arange(N)] * 3), indexing="ij"), axis=-1).reshape(-1, 3) + 0.5) / N
        inside = np.zeros(len(f), dtype=bool)
        sh = np.stack(np.meshgrid(*([np.arange(-1, 2)] * 3), indexing="ij"), axis=-1).reshape(-1, 3)
        for t, R in zip(p.tau, p.radii):
            for s in sh:
                inside |= np.linalg.norm((f - t - s) @ p.A, axis=1) < R
        m = (~inside).astype(np.float64)
        ax = np.arange(-2, 3)
        g = np.stack(np.meshgrid(ax, ax, ax, indexing="ij"), axis=-1).reshape(-1, 3)
        dft = (np.exp(2j * np.pi * (g @ f.T)) @ m / len(f)).reshape(5, 5, 5)
        errs.append(np.abs(dft - th).max())
    assert errs[1] < 6e-3 and errs[1] < 0.75 * errs[0], errs
