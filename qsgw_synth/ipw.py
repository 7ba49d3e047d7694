"""Seeded inputs for the interstitial-plane-wave (IPW) block of the matrix elements (Eqs. 4-5 and 8,
PAPER.md:106-110,130).  Input generation only: a lattice, non-overlapping muffin-tin spheres, the integer reciprocal
vectors of the three plane-wave sets, the Fourier coefficients of the interstitial indicator function on the integer box
the kernel looks differences up in, and random plane-wave coefficients of the eigenfunctions.  No z is computed here.

Stand-in for what a PMT/LAPW code provides (ecalj's IPW lists and its step-function coefficients); recipe in DESIGN.md 4f.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

from .configs import BASE_SEED


@dataclass
class IpwProblem:
    A: np.ndarray            # (3, 3) lattice vectors, rows, bohr
    tau: np.ndarray          # (S, 3) sphere centres, fractional
    radii: np.ndarray        # (S,)   muffin-tin radii, bohr
    kappa_kq: np.ndarray     # fractional crystal momenta with kappa_kq + kappa_ipw = kappa_k (reciprocal-lattice units)
    kappa_ipw: np.ndarray
    kappa_k: np.ndarray
    g_kq: np.ndarray         # int32 (N_kq, 3)  plane waves of the eigenfunctions on the conjugated side (bands n')
    g_k: np.ndarray          # int32 (N_k, 3)   plane waves of the eigenfunctions on the other side (bands n)
    g_ipw: np.ndarray        # int32 (N_ipw, 3) IPWs of the mixed product basis
    L: np.ndarray            # int32 (3,) half extents of the theta box: every g_k - g_kq - g_ipw lies inside
    theta: np.ndarray        # complex128 (2 L0 + 1, 2 L1 + 1, 2 L2 + 1): theta[g + L]
    Bkq: np.ndarray          # complex128 (n_u, N_kq)  beta^{n'}_G
    Bk: np.ndarray           # complex128 (n_o, N_k)   beta^{n}_G


def recip(A: np.ndarray) -> np.ndarray:
    """Rows = reciprocal lattice vectors b_i, a_i . b_j = 2 pi delta_ij."""
    return 2.0 * np.pi * np.linalg.inv(A).T


def g_sphere(Bm: np.ndarray, kappa: np.ndarray, cutoff: float) -> np.ndarray:
    """All integer g with |(g + kappa) . B|^2 <= cutoff (Ry), ordered by length then lexicographically."""
    n = int(np.ceil(np.sqrt(cutoff) / np.min(np.linalg.svd(Bm, compute_uv=False)))) + 1
    r = np.arange(-n, n + 1)
    g = np.stack(np.meshgrid(r, r, r, indexing="ij"), axis=-1).reshape(-1, 3)
    q2 = np.sum(((g + kappa) @ Bm) ** 2, axis=1)
    keep = q2 <= cutoff
    g, q2 = g[keep], q2[keep]
    order = np.lexsort((g[:, 2], g[:, 1], g[:, 0], np.round(q2, 9)))
    return g[order].astype(np.int32)


def interstitial_theta(A: np.ndarray, tau: np.ndarray, radii: np.ndarray, L: np.ndarray) -> np.ndarray:
    """theta(g) = (1/Omega) int_cell Theta_I(r) exp(i G.r) d^3r, G = g . B, for every integer g in the box [-L, L]:
    theta(0) = 1 - sum_s 4 pi R_s^3 / (3 Omega);  theta(g) = - sum_s (4 pi R_s^3 / Omega) j1(|G| R_s) / (|G| R_s) exp(i G.tau_s)."""
    Bm = recip(A)
    vol = abs(np.linalg.det(A))
    ax = [np.arange(-int(l), int(l) + 1) for l in L]
    g = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).astype(np.float64)      # (.., 3)
    G = g @ Bm
    Gn = np.linalg.norm(G, axis=-1)
    th = np.zeros(Gn.shape, dtype=np.complex128)
    for t, R in zip(tau, radii):
        x = Gn * R
        with np.errstate(divide="ignore", invalid="ignore"):
            f = np.where(x > 1e-6, (np.sin(x) - x * np.cos(x)) / x ** 3, 1.0 / 3.0 - x * x / 30.0)
        th -= (4.0 * np.pi * R ** 3 / vol) * f * np.exp(2j * np.pi * (g @ t))
    th[tuple(int(l) for l in L)] += 1.0
    return th


def synthetic_ipw(n_o: int = 8, n_u: int = 12, cut_pw: float = 3.0, cut_ipw: float = 4.0, n_spheres: int = 2,
                  a0: float = 7.5, seed: int = 0) -> IpwProblem:
    """cut_pw ~ the paper's 3 Ry APW cutoff; a0 = lattice constant scale in bohr (sets the counts)."""
    rng = np.random.default_rng(BASE_SEED + 7000 + seed)
    A = a0 * (np.eye(3) + 0.06 * rng.standard_normal((3, 3)))
    tau = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5], [0.25, 0.75, 0.5], [0.75, 0.25, 0.0]])[:n_spheres] \
        + 0.02 * rng.standard_normal((n_spheres, 3))
    # radii: 0.40-0.45 of the distance to the nearest other sphere centre (periodic images included): touching-free spheres
    sh = np.stack(np.meshgrid(*([np.arange(-1, 2)] * 3), indexing="ij"), axis=-1).reshape(-1, 3)
    dmin = np.full(n_spheres, np.inf)
    for i in range(n_spheres):
        for j in range(n_spheres):
            d = np.linalg.norm((tau[j] - tau[i] + sh) @ A, axis=1)
            d = d[d > 1e-9]
            dmin[i] = min(dmin[i], d.min())
    radii = dmin * (0.40 + 0.05 * rng.random(n_spheres))
    Bm = recip(A)
    kappa_kq = rng.random(3) - 0.5
    kappa_ipw = rng.random(3) - 0.5
    kappa_k = kappa_kq + kappa_ipw                               # umklapp stays in kappa_k: only integer differences matter
    g_kq = g_sphere(Bm, kappa_kq, cut_pw)
    g_k = g_sphere(Bm, kappa_k, cut_pw)
    g_ipw = g_sphere(Bm, kappa_ipw, cut_ipw)
    d_hi = g_k.max(0) - g_kq.min(0) - g_ipw.min(0)
    d_lo = g_k.min(0) - g_kq.max(0) - g_ipw.max(0)
    L = np.maximum(np.abs(d_hi), np.abs(d_lo)).astype(np.int32)
    theta = interstitial_theta(A, tau, radii, L)

    def coeffs(n, g, kappa):
        q2 = np.sum(((g + kappa) @ Bm) ** 2, axis=1)
        c = (rng.standard_normal((n, len(g))) + 1j * rng.standard_normal((n, len(g)))) * np.exp(-0.25 * q2)[None, :]
        return c / np.linalg.norm(c, axis=1, keepdims=True)

    Bkq = coeffs(n_u, g_kq, kappa_kq)
    Bk = coeffs(n_o, g_k, kappa_k)
    return IpwProblem(A, tau, radii, kappa_kq, kappa_ipw, kappa_k, g_kq, g_k, g_ipw, L, theta, Bkq, Bk)
