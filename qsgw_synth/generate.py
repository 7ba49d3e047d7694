"""Seeded input generator (NumPy only; no method arithmetic).

Draw order: P, then per (spin, k): unitary for k, unitary for
k+q, eps_k, eps_{k+q}.  Seed = 250603477 + config index (+ optional offset).

Layouts returned are the boundary layouts of include/qsgw.h:
  P      complex128 [sum_s m_s*b_s*b_s], site-major, each site [I][alpha][beta]
  Ck     complex128 [n_k][n_o][N_b]   (row = band, i.e. column-major N_b x n_o)
  Ckq    complex128 [n_k][n_u][N_b]
  eps_k, f_k   float64 [n_k][n_o];  eps_kq, f_kq  float64 [n_k][n_u]
  omega  float64 [n_freq]
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List

import numpy as np

from .configs import BASE_SEED, WorkloadConfig


def haar_unitary(rng: np.random.Generator, n: int) -> np.ndarray:
    """Haar-distributed n x n unitary: QR of a complex Ginibre matrix with the
    diag(R)/|diag(R)| phase fix."""
    g = (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) / np.sqrt(2.0)
    q, r = np.linalg.qr(g)
    d = np.diagonal(r)
    return q * (d / np.abs(d))[None, :]


def omega_grid(cfg: WorkloadConfig) -> np.ndarray:
    """omega_0 = 0, then geometric from omega_1 to omega_max (n_freq points in all)."""
    om = np.zeros(cfg.n_freq)
    if cfg.n_freq > 1:
        if cfg.n_freq == 2:
            om[1] = cfg.omega_max
        else:
            om[1:] = np.geomspace(cfg.omega_1, cfg.omega_max, cfg.n_freq - 1)
    return om


@dataclass
class SpinChannel:
    Ck: np.ndarray
    Ckq: np.ndarray
    eps_k: np.ndarray
    f_k: np.ndarray
    eps_kq: np.ndarray
    f_kq: np.ndarray


@dataclass
class Problem:
    cfg: WorkloadConfig
    P: np.ndarray            # flat, site-major
    omega: np.ndarray
    spins: List[SpinChannel]

    def P_site(self, s: int) -> np.ndarray:
        b, m = self.cfg.orb_per_site, self.cfg.pb_per_site
        off = sum(mm * bb * bb for bb, mm in zip(b[:s], m[:s]))
        return self.P[off: off + m[s] * b[s] * b[s]].reshape(m[s], b[s], b[s])


def _fermi(eps: np.ndarray, kT: float) -> np.ndarray:
    x = np.clip(eps / kT, -700.0, 700.0)
    return 1.0 / (1.0 + np.exp(x))


def generate(cfg: WorkloadConfig, seed_offset: int = 0, n_k: int | None = None) -> Problem:
    """Generate the seeded problem.  `n_k` truncates the k loop (same stream prefix,
    so the first n_k k-points equal those of the full problem)."""
    rng = np.random.default_rng(BASE_SEED + cfg.index + seed_offset)
    nk = cfg.n_k if n_k is None else n_k
    nb = cfg.n_b
    parts = []
    for b, m in zip(cfg.orb_per_site, cfg.pb_per_site):
        sd = np.sqrt(0.5 / b)   # E|P|^2 = 1/b_s
        parts.append((sd * (rng.standard_normal((m, b, b)) +
                            1j * rng.standard_normal((m, b, b)))).reshape(-1))
    P = np.concatenate(parts)
    spins = []
    for _ in range(cfg.n_spin):
        Ck = np.empty((nk, cfg.n_o, nb), dtype=np.complex128)
        Ckq = np.empty((nk, cfg.n_u, nb), dtype=np.complex128)
        eps_k = np.empty((nk, cfg.n_o)); f_k = np.empty((nk, cfg.n_o))
        eps_kq = np.empty((nk, cfg.n_u)); f_kq = np.empty((nk, cfg.n_u))
        for k in range(nk):
            Uk = haar_unitary(rng, nb)
            Ukq = haar_unitary(rng, nb)
            if cfg.kind == "insulator":
                o0, u0 = 0, cfg.n_o
                e_o = np.sort(rng.uniform(*cfg.eps_occ, cfg.n_o))
                e_u = np.sort(rng.uniform(*cfg.eps_unocc, cfg.n_u))
                fo, fu = np.ones(cfg.n_o), np.zeros(cfg.n_u)
            else:
                o0, u0 = cfg.o_first, cfg.u_first
                ek_all = np.sort(rng.uniform(*cfg.eps_all, nb))
                ekq_all = np.sort(rng.uniform(*cfg.eps_all, nb))
                e_o = ek_all[o0:o0 + cfg.n_o]
                e_u = ekq_all[u0:u0 + cfg.n_u]
                fo, fu = _fermi(e_o, cfg.kT), _fermi(e_u, cfg.kT)
            # column n of the unitary = band n; stored band-major (row = band)
            Ck[k] = Uk[:, o0:o0 + cfg.n_o].T
            Ckq[k] = Ukq[:, u0:u0 + cfg.n_u].T
            eps_k[k], f_k[k], eps_kq[k], f_kq[k] = e_o, fo, e_u, fu
        spins.append(SpinChannel(Ck, Ckq, eps_k, f_k, eps_kq, f_kq))
    return Problem(cfg=cfg, P=P, omega=omega_grid(cfg), spins=spins)


def coulomb_eigenvalues(cfg: WorkloadConfig, seed_offset: int = 0) -> np.ndarray:
    """Synthetic Coulomb eigenvalues v_mu > 0 of the product basis (inputs of Eqs. 10/19):
    a 4 pi / |q+G|^2-like decaying spectrum, v_mu = 4 pi / (0.3 + 0.05 mu) Ha, jittered by a seeded factor in
    [0.8, 1.25] and shuffled over the product functions.  The paper's real v_mu(q) come from its Coulomb-matrix
    diagonalisation (Eq. 7), which needs data only a full code provides; these keep the dynamic range (~1e2)."""
    rng = np.random.default_rng(BASE_SEED + 1000 + cfg.index + seed_offset)
    mu = np.arange(cfg.n_m, dtype=np.float64)
    v = 4.0 * np.pi / (0.3 + 0.05 * mu) * np.exp(rng.uniform(np.log(0.8), np.log(1.25), cfg.n_m))
    return rng.permutation(v)


def synthetic_wc(n_m: int, omega: np.ndarray, seed: int = 0, hermitian: bool = True) -> np.ndarray:
    """Synthetic screened interaction W^c(i omega_i), complex128 [n_freq][n_m][n_m] (an INPUT of Eq. 22,
    PAPER.md:197-205, where the paper reads it from the W task): negative semidefinite Hermitian matrices with
    monotonic damping along the imaginary axis, W_i = -(G_i G_i^H) / (n_m (1 + omega_i^2)) with
    G_i = G + 0.3 H_i complex Gaussian.  hermitian=False adds a general complex part (tests that must tell W from
    its transpose)."""
    rng = np.random.default_rng(BASE_SEED + 2000 + seed)
    c = lambda *sh: (rng.standard_normal(sh) + 1j * rng.standard_normal(sh)) / np.sqrt(2.0)
    G = c(n_m, n_m)
    out = np.empty((len(omega), n_m, n_m), dtype=np.complex128)
    for i, w in enumerate(np.asarray(omega, dtype=np.float64)):
        Gi = G + 0.3 * c(n_m, n_m)
        out[i] = -(Gi @ Gi.conj().T) / (n_m * (1.0 + w * w))
        if not hermitian:
            out[i] += 0.2 * c(n_m, n_m) / (1.0 + w * w)
    return out


def log_bin_edges(n_bins: int, w_first: float = 1e-3, w_max: float = 2.5) -> np.ndarray:
    """Edges of the logarithmic histogram mesh on the real axis ("omega_j = 1e-5 x 1.03^j Ry ... ~100
    mesh points"): n_bins + 1 geometric edges from w_first > 0 to w_max (Ha)."""
    return np.geomspace(w_first, w_max, n_bins + 1)


def binned_pair_weights(eps_k, f_k, eps_kq, f_kq, edges, rel_width: float = 0.05, occ_tol: float = 1e-12):
    """Synthetic stand-in for the tetrahedron weights w(n', n, k, bin) of Eqs. (16)-(17), which
    the paper computes on the CPU before the accumulation loop (Alg. 1 line 8) and which are INPUTS of the binned
    accumulation: every kept pair (f_n (1 - f_n') > occ_tol, D = eps_kq[n'] - eps_k[n] > 0) spreads its occupation
    factor f_n (1 - f_n') uniformly over the energy window [D (1 - rel_width), D (1 + rel_width)] -- the stand-in
    for the band dispersion inside a tetrahedron -- and a bin receives the fraction of the window it overlaps.
    Returns the CSR-by-bin triple (bin_ptr int32 [n_bins+1], pair int32 [nnz] = n * n_u + n', w float64 [nnz]);
    the part of a window outside [edges[0], edges[-1]) is dropped."""
    eps_k = np.asarray(eps_k); eps_kq = np.asarray(eps_kq)
    edges = np.asarray(edges, dtype=np.float64)
    n_o, n_u = len(eps_k), len(eps_kq)
    D = eps_kq[None, :] - eps_k[:, None]
    occ = np.asarray(f_k)[:, None] * (1.0 - np.asarray(f_kq)[None, :])
    keep = (occ > occ_tol) & (D > 0)
    n_idx, u_idx = np.nonzero(keep)
    lo = D[keep] * (1.0 - rel_width)
    hi = D[keep] * (1.0 + rel_width)
    wgt = occ[keep]
    pidx = (n_idx * n_u + u_idx).astype(np.int32)
    j_lo = np.clip(np.searchsorted(edges, lo, side="right") - 1, 0, len(edges) - 2)
    j_hi = np.clip(np.searchsorted(edges, hi, side="left") - 1, 0, len(edges) - 2)
    bins, pairs, ws = [], [], []
    for off in range(int((j_hi - j_lo).max()) + 1 if len(lo) else 0):
        j = j_lo + off
        sel = j <= j_hi
        ov = np.minimum(hi[sel], edges[j[sel] + 1]) - np.maximum(lo[sel], edges[j[sel]])
        ok = ov > 0
        bins.append(j[sel][ok]); pairs.append(pidx[sel][ok]); ws.append(wgt[sel][ok] * ov[ok] / (hi[sel][ok] - lo[sel][ok]))
    if bins:
        bins = np.concatenate(bins); pairs = np.concatenate(pairs); ws = np.concatenate(ws)
    else:
        bins = np.zeros(0, dtype=np.int64); pairs = np.zeros(0, dtype=np.int32); ws = np.zeros(0)
    order = np.lexsort((pairs, bins))
    bin_ptr = np.zeros(len(edges), dtype=np.int32)
    np.add.at(bin_ptr, bins + 1, 1)
    return np.cumsum(bin_ptr).astype(np.int32), pairs[order].astype(np.int32), ws[order].astype(np.float64)


def synthetic_mpb_matrices(n_m: int, seed: int = 0, cond_o: float = 50.0, kappa: float = 0.05):
    """Overlap and Coulomb matrices of a non-orthogonal mixed product basis (inputs of the generalized eigenproblem,
    PAPER.md:116-118): M = E S with a seeded non-unitary S (condition number ~ cond_o: IPWs are not orthogonal), so
    O = S^H S and v = S^H diag(lambda) S, lambda_mu = 4 pi / (|q_mu|^2 + kappa^2) on seeded |q_mu| (the plane-wave form
    of the Coulomb interaction with the paper's exp(-kappa r) regularisation).  Returns (v, O, lambda sorted
    descending): the generalized eigenvalues of (v, O) are lambda by construction."""
    rng = np.random.default_rng(BASE_SEED + 9000 + seed)
    Q1, Q2 = haar_unitary(rng, n_m), haar_unitary(rng, n_m)
    sv = np.exp(np.linspace(0.0, np.log(cond_o), n_m))
    S = (Q1 * sv[None, :]) @ Q2
    qn = np.concatenate([[0.02], np.sort(rng.uniform(0.3, 6.0, n_m - 1))]) if n_m > 1 else np.array([0.02])
    lam = 4.0 * np.pi / (qn ** 2 + kappa ** 2)
    O = S.conj().T @ S
    v = S.conj().T @ (lam[:, None] * S)
    O = 0.5 * (O + O.conj().T)
    v = 0.5 * (v + v.conj().T)
    return v, O, np.sort(lam)[::-1]
