"""Pins of the oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formula or re-call its routine on the same path:
brute-force literal loops, complex two-fraction form of Eq. 14, closed forms in
limits, completeness of a unitary, gauge invariances, ZHERK / matmul reductions.
"""
import numpy as np
import pytest
import scipy.linalg

import oracle
from qsgw_synth import CONFIGS, WorkloadConfig, generate, get_config, haar_unitary, scaled_config


def _sites(prob):
    return [prob.P_site(s) for s in range(prob.cfg.n_sites)]


def _chi(prob, spin=0, **kw):
    sp = prob.spins[spin]
    return oracle.chi0_ref(_sites(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                           kw.pop("omega", prob.omega), **kw)


def tiny_cfg(kind="insulator", **kw):
    base = dict(name="tiny", index=90, orb_per_site=(2, 3), pb_per_site=(3, 2), n_k=2, n_spin=1,
                n_o=2, n_u=3, n_freq=3, kind=kind, eps_occ=(-0.45, 0.0), eps_unocc=(0.02, 1.1))
    base.update(kw)
    return WorkloadConfig(**base)


# ---- pin 1: brute force (literal 7-loop) on tiny ragged-site inputs ------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_bruteforce_tiny(seed):
    prob = generate(tiny_cfg(), seed_offset=seed)
    sp = prob.spins[0]
    fast = _chi(prob)
    naive = oracle.chi0_ref_naive(_sites(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                                  sp.f_kq, prob.omega)
    assert np.abs(fast - naive).max() <= 1e-13 * max(1.0, np.abs(naive).max())


def test_bruteforce_tiny_metal_fractional_occupations():
    cfg = tiny_cfg(kind="metal", orb_per_site=(3, 3), pb_per_site=(2, 3), n_o=3, n_u=4,
                   eps_all=(-0.01, 0.01), o_first=0, u_first=2, kT=5e-3, index=91)
    prob = generate(cfg)
    sp = prob.spins[0]
    assert ((sp.f_k > 0.01) & (sp.f_k < 0.99)).any()      # genuinely fractional
    fast = _chi(prob)
    naive = oracle.chi0_ref_naive(_sites(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                                  sp.f_kq, prob.omega)
    assert np.abs(fast - naive).max() <= 1e-13 * max(1.0, np.abs(naive).max())


# ---- pin 2: weight = bracket of Eq. 14 in complex arithmetic -------
def test_weight_is_eq14_bracket_on_imaginary_axis():
    rng = np.random.default_rng(7)
    eps_k = -rng.uniform(0.01, 0.5, 5); eps_kq = rng.uniform(0.01, 1.0, 6)
    f_k = np.ones(5); f_kq = np.zeros(6)
    omega = np.array([0.0, 1e-3, 0.3, 2.0, 20.0])
    w = oracle.pair_weights(eps_k, f_k, eps_kq, f_kq, omega)
    for j, om in enumerate(omega):
        for n in range(5):
            for m in range(6):
                D = eps_kq[m] - eps_k[n]
                br = 1.0 / (1j * om - D) - 1.0 / (1j * om + D)
                assert abs(br.imag) < 1e-12 * abs(br.real)
                assert w[j, n, m] == pytest.approx(br.real, rel=1e-13)
    # even in omega (Pi(w) = Pi(-w))
    w_neg = oracle.pair_weights(eps_k, f_k, eps_kq, f_kq, -omega)
    assert np.array_equal(w, w_neg)


def test_weight_occupation_filter_and_zero_over_zero():
    eps_k = np.array([0.0, -0.1]); eps_kq = np.array([0.0, 0.2])
    f_k = np.array([0.5, 1.0]); f_kq = np.array([0.5, 1.0 - 1e-13])
    w = oracle.pair_weights(eps_k, f_k, eps_kq, f_kq, np.array([0.0, 1.0]))
    assert w[0, 0, 0] == 0.0            # D = 0 and omega = 0: dropped (reading R3)
    assert w[1, 0, 0] == 0.0            # D = 0: numerator zero
    assert np.all(w[:, :, 1] == 0.0)    # f(1-f') = 1e-13 <= 1e-12: dropped (reading R2)
    assert w[0, 1, 0] == pytest.approx(-2.0 * 0.5 / 0.1)
    # partially filled pair with D < 0 is kept with a positive weight (reading R4)
    w2 = oracle.pair_weights(np.array([0.001]), np.array([0.4]), np.array([-0.001]),
                             np.array([0.6]), np.array([0.0]))
    assert w2[0, 0, 0] == pytest.approx(-2 * 0.4 * 0.4 * (-0.002) / (0.002 ** 2)) and w2[0, 0, 0] > 0


# ---- pins 3/4: Hermitian, negative semidefinite, monotone decay ----
@pytest.mark.parametrize("idx", [0, 1])
def test_hermitian_negative_monotone(idx):
    cfg = get_config(idx)
    prob = generate(cfg, n_k=min(cfg.n_k, 6))
    chi = _chi(prob)
    nrm = np.linalg.norm(chi, axis=(1, 2))
    for j in range(cfg.n_freq):
        assert np.linalg.norm(chi[j] - chi[j].conj().T) <= 1e-14 * nrm[j]
        ev = np.linalg.eigvalsh(0.5 * (chi[j] + chi[j].conj().T))
        assert ev.max() <= 1e-12 * abs(ev.min())           # negative (semi)definite
    for j in range(cfg.n_freq - 1):
        d = chi[j + 1] - chi[j]
        ev = np.linalg.eigvalsh(0.5 * (d + d.conj().T))
        assert ev.min() >= -1e-12 * nrm[j]                  # Loewner-monotone towards 0
        assert nrm[j + 1] < nrm[j]
        assert np.all(np.diagonal(chi[j + 1]).real >= np.diagonal(chi[j]).real)
    assert np.all(np.diagonal(chi[-1]).real < 0)


def test_metal_sign_split():
    """cfg-2 shape (reduced k): D>0 part is NSD, D<0 part is PSD (reading R4)."""
    cfg = scaled_config(get_config(2), n_k=3, n_spin=1)
    prob = generate(cfg)
    sp = prob.spins[0]
    sites = _sites(prob)
    n_m = cfg.n_m
    neg = np.zeros((cfg.n_freq, n_m, n_m), complex); pos = np.zeros_like(neg)
    n_negD = 0
    for k in range(cfg.n_k):
        z = oracle.zmel_ref(sites, sp.Ck[k], sp.Ckq[k])
        w = oracle.pair_weights(sp.eps_k[k], sp.f_k[k], sp.eps_kq[k], sp.f_kq[k], prob.omega)
        n_negD += int((w[0] > 0).sum())
        oracle.chi0_accumulate_ref(neg, z, np.minimum(w, 0.0))
        oracle.chi0_accumulate_ref(pos, z, np.maximum(w, 0.0))
    for j in range(cfg.n_freq):
        assert np.linalg.eigvalsh(neg[j]).max() <= 1e-10
        assert np.linalg.eigvalsh(pos[j]).min() >= -1e-10
    total = _chi(prob)
    assert np.allclose((neg + pos) / cfg.n_k, total, rtol=0, atol=1e-12 * np.abs(total).max())


# ---- pins 5/6: closed forms at omega -> infinity and omega = 0 -------------------------
def test_static_and_tail_closed_forms():
    cfg = scaled_config(get_config(0), n_k=3)
    prob = generate(cfg)
    sp = prob.spins[0]
    sites = _sites(prob)
    n_m = cfg.n_m
    big = 1.0e4
    chi = _chi(prob, omega=np.array([0.0, 20.0, big]))
    stat = np.zeros((n_m, n_m), complex); tail = np.zeros_like(stat)
    dmax = 0.0
    for k in range(cfg.n_k):
        Z = oracle.zmel_ref(sites, sp.Ck[k], sp.Ckq[k]).reshape(-1, n_m)
        D = (sp.eps_kq[k][None, :] - sp.eps_k[k][:, None]).reshape(-1)
        dmax = max(dmax, D.max())
        stat += -2.0 * (Z.conj().T / D) @ Z
        tail += -2.0 * (Z.conj().T * D) @ Z
    stat /= cfg.n_k; tail /= cfg.n_k
    assert np.linalg.norm(chi[0] - stat) <= 1e-13 * np.linalg.norm(stat)
    dev = np.linalg.norm(big ** 2 * chi[2] - tail) / np.linalg.norm(tail)
    assert dev <= (dmax / big) ** 2
    # omega = 20 Ha is NOT in the tail (SURVEY c.3-5): deviation is ~1e-3, bounded by (D/omega)^2
    dev20 = np.linalg.norm(400.0 * chi[1] - tail) / np.linalg.norm(tail)
    assert 1e-5 < dev20 <= (dmax / 20.0) ** 2


# ---- pin 7: completeness of the unitary pins stage (a) independently -------------------
def test_completeness_sum_over_all_unoccupied():
    rng = np.random.default_rng(11)
    b = (3, 4); m = (2, 5); nb = sum(b)
    P = [rng.standard_normal((mm, bb, bb)) + 1j * rng.standard_normal((mm, bb, bb))
         for bb, mm in zip(b, m)]
    Ck = haar_unitary(rng, nb)[:, :3].T.copy()          # 3 occupied-side bands
    Ckq = haar_unitary(rng, nb).T.copy()                # ALL columns of a unitary
    z = oracle.zmel_ref(P, Ck, Ckq)                     # (3, nb, n_m)
    G = np.einsum("npi,npj->nij", z.conj(), z)          # sum over n' with unit weights
    ob = np.concatenate([[0], np.cumsum(b)]); om = np.concatenate([[0], np.cumsum(m)])
    for n in range(3):
        for s in range(2):
            T = np.einsum("iab,b->ia", P[s], Ck[n, ob[s]:ob[s + 1]])
            ref = T.conj() @ T.T                        # sum_alpha conj(T_I) T_J
            got = G[n, om[s]:om[s + 1], om[s]:om[s + 1]]
            assert np.allclose(got, ref, rtol=0, atol=1e-12 * np.abs(ref).max())
        cross = G[n, om[0]:om[1], om[1]:om[2]]
        assert np.abs(cross).max() <= 1e-13 * np.abs(G[n]).max()   # exactly 0 across sites


def test_zmel_single_term_orientation():
    """One non-zero coefficient each: z = conj(Ckq[a,n']) P[I,a,b] Ck[b,n] -- catches a
    transposed P, a missing conjugate or swapped k / k+q."""
    b = (2, 3); m = (2, 2)
    rng = np.random.default_rng(3)
    P = [rng.standard_normal((mm, bb, bb)) + 1j * rng.standard_normal((mm, bb, bb))
         for bb, mm in zip(b, m)]
    Ck = np.zeros((1, 5), complex); Ckq = np.zeros((1, 5), complex)
    Ck[0, 2 + 1] = 0.3 - 0.7j         # site 1, beta = 1
    Ckq[0, 2 + 2] = -0.5 + 0.2j       # site 1, alpha = 2
    z = oracle.zmel_ref(P, Ck, Ckq)
    assert np.all(z[0, 0, :2] == 0)
    for I in range(2):
        assert z[0, 0, 2 + I] == pytest.approx(np.conj(Ckq[0, 4]) * P[1][I, 2, 1] * Ck[0, 3])


# ---- pin 8: gauge invariance, |c|^2 scaling, permutation invariance --------------------
def test_gauge_scaling_permutation():
    cfg = scaled_config(get_config(0), n_k=3)
    prob = generate(cfg)
    sp = prob.spins[0]
    ref = _chi(prob)
    rng = np.random.default_rng(5)
    ph_o = np.exp(2j * np.pi * rng.random((cfg.n_k, cfg.n_o, 1)))
    ph_u = np.exp(2j * np.pi * rng.random((cfg.n_k, cfg.n_u, 1)))
    sites = _sites(prob)
    g = oracle.chi0_ref(sites, sp.Ck * ph_o, sp.Ckq * ph_u, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                        prob.omega)
    assert np.linalg.norm(g - ref) <= 1e-13 * np.linalg.norm(ref)
    c = 0.7 - 1.9j
    s = oracle.chi0_ref([c * p for p in sites], sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                        sp.f_kq, prob.omega)
    assert np.linalg.norm(s - abs(c) ** 2 * ref) <= 1e-13 * np.linalg.norm(ref)
    perm = rng.permutation(cfg.n_k)
    po = rng.permutation(cfg.n_o); pu = rng.permutation(cfg.n_u)
    p = oracle.chi0_ref(sites, sp.Ck[perm][:, po], sp.Ckq[perm][:, pu], sp.eps_k[perm][:, po],
                        sp.f_k[perm][:, po], sp.eps_kq[perm][:, pu], sp.f_kq[perm][:, pu],
                        prob.omega)
    assert np.linalg.norm(p - ref) <= 1e-13 * np.linalg.norm(ref)


def test_degenerate_subspace_rotation():
    cfg = scaled_config(get_config(0), n_k=2)
    prob = generate(cfg)
    sp = prob.spins[0]
    eps_k = sp.eps_k.copy(); eps_k[:, 1] = eps_k[:, 0]; eps_k[:, 2] = eps_k[:, 0]  # 3-fold degenerate
    sites = _sites(prob)
    ref = oracle.chi0_ref(sites, sp.Ck, sp.Ckq, eps_k, sp.f_k, sp.eps_kq, sp.f_kq, prob.omega)
    rng = np.random.default_rng(9)
    Ck = sp.Ck.copy()
    for k in range(cfg.n_k):
        R = haar_unitary(rng, 3)
        Ck[k, :3, :] = R.T @ sp.Ck[k, :3, :]
    rot = oracle.chi0_ref(sites, Ck, sp.Ckq, eps_k, sp.f_k, sp.eps_kq, sp.f_kq, prob.omega)
    assert np.linalg.norm(rot - ref) <= 1e-13 * np.linalg.norm(ref)


# ---- pin 9: library reductions (ZHERK) --------------------------------------------------
def test_zherk_reduction():
    cfg = scaled_config(get_config(0), n_k=2)
    prob = generate(cfg)
    sp = prob.spins[0]
    sites = _sites(prob)
    chi = _chi(prob)
    n_m = cfg.n_m
    for j in (0, 3, cfg.n_freq - 1):
        acc = np.zeros((n_m, n_m), complex)
        for k in range(cfg.n_k):
            Z = oracle.zmel_ref(sites, sp.Ck[k], sp.Ckq[k]).reshape(-1, n_m)
            D = (sp.eps_kq[k][None, :] - sp.eps_k[k][:, None]).reshape(-1)
            Y = np.sqrt(2.0 * D / (D * D + prob.omega[j] ** 2))[:, None] * Z
            up = scipy.linalg.blas.zherk(1.0, Y, trans=2, lower=0)    # Y^H Y, upper triangle
            acc += np.triu(up) + np.triu(up, 1).conj().T
        assert np.linalg.norm(chi[j] + acc / cfg.n_k) <= 1e-13 * np.linalg.norm(chi[j])


# ---- pin 10: one-pair scalar case ---------------------------------------------------------
def test_one_pair_scalar():
    P = [np.array([[[0.5 - 1.5j]]])]
    Ck = np.array([[[0.6 + 0.8j]]]); Ckq = np.array([[[-0.28 + 0.96j]]])
    eps_k = np.array([[-0.2]]); eps_kq = np.array([[0.3]])
    f_k = np.array([[1.0]]); f_kq = np.array([[0.0]])
    om = np.array([0.0, 0.5])
    chi = oracle.chi0_ref(P, Ck, Ckq, eps_k, f_k, eps_kq, f_kq, om)
    zabs2 = abs(0.5 - 1.5j) ** 2       # |Ck| = |Ckq| = 1
    assert chi[0, 0, 0] == pytest.approx(-2 * 0.5 / 0.25 * zabs2)
    assert chi[1, 0, 0] == pytest.approx(-2 * 0.5 / 0.5 * zabs2)


# ---- sketch / sampled-entry / finalize helpers agree with the full matrix ----------------
def test_sketch_entries_finalize_consistent():
    cfg = scaled_config(get_config(0), n_k=2)
    prob = generate(cfg)
    sp = prob.spins[0]
    sites = _sites(prob)
    chi = _chi(prob)
    rng = np.random.default_rng(1)
    V = rng.standard_normal((cfg.n_m, 4)) + 1j * rng.standard_normal((cfg.n_m, 4))
    S = oracle.chi0_sketch_ref(sites, sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                               prob.omega, V)
    assert np.linalg.norm(S - chi @ V) <= 1e-13 * np.linalg.norm(S)
    rows = rng.integers(0, cfg.n_m, 9); cols = rng.integers(0, cfg.n_m, 9)
    E = oracle.chi0_entries_ref(sites, sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                                prob.omega, rows, cols)
    assert np.allclose(E, chi[:, rows, cols], rtol=0, atol=1e-13 * np.abs(chi).max())
    H = oracle.hermitian_finalize_ref(chi)
    assert np.linalg.norm(H - chi) <= 1e-14 * np.linalg.norm(chi)
    assert np.all(np.diagonal(H, axis1=1, axis2=2).imag == 0)


# ---- generator sanity (shapes / recipe; no method arithmetic) ------------------------------
def test_generator_recipe():
    for cfg in CONFIGS:
        prob = generate(cfg, n_k=1)
        sp = prob.spins[0]
        assert len(prob.spins) == cfg.n_spin
        assert sp.Ck.shape == (1, cfg.n_o, cfg.n_b) and sp.Ckq.shape == (1, cfg.n_u, cfg.n_b)
        assert np.allclose(sp.Ck[0].conj() @ sp.Ck[0].T, np.eye(cfg.n_o), atol=1e-12)
        assert prob.omega[0] == 0.0 and prob.omega[-1] == pytest.approx(20.0)
        assert np.all(np.diff(prob.omega) > 0)
        assert np.all(np.diff(sp.eps_k[0]) >= 0) and np.all(np.diff(sp.eps_kq[0]) >= 0)
        v = np.mean(np.abs(prob.P_site(0)) ** 2) * cfg.orb_per_site[0]
        assert 0.9 < v < 1.1
    p2 = generate(get_config(2), n_k=2)
    f = p2.spins[0].f_k
    assert f.min() >= 0 and f.max() <= 1
    assert ((f > 1e-6) & (f < 1 - 1e-6)).any()          # the metal has partially filled bands (kT = 1e-3 Ha)
    full = generate(get_config(0)); part = generate(get_config(0), n_k=3)
    assert np.array_equal(full.spins[0].Ck[:3], part.spins[0].Ck)


def test_table2_z_size_bookkeeping():
    """Z_size = n_pb * n_all * n_qp * 16 B reproduces Table 2."""
    import os
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden",
            "table2_zsize.txt")) if l.strip() and not l.startswith("#")]
    for name, n_pb, n_all, n_qp, gib in rows:
        got = int(n_pb) * int(n_all) * int(n_qp) * 16 / 2.0 ** 30
        assert got == pytest.approx(float(gib), abs=0.006), name
