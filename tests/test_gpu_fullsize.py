"""Full-size parity (the launch configuration bench.py times): sampled entries and the exact
sketch chi0 @ V computed by the oracle without forming chi0."""
import numpy as np
import pytest

import oracle
from qsgw_synth import generate, get_config
from gpu_helpers import run_cuda, sites_of

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def _sampled_and_sketch(prob, spin, got, tol):
    cfg = prob.cfg
    sp = prob.spins[spin]
    rng = np.random.default_rng(1234 + cfg.index)
    n_m = cfg.n_m
    V = (rng.standard_normal((n_m, 4)) + 1j * rng.standard_normal((n_m, 4))) / np.sqrt(2)
    S = oracle.chi0_sketch_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                               prob.omega, V, occ_tol=cfg.occ_tol)
    num = np.linalg.norm((got @ V - S).reshape(len(prob.omega), -1), axis=1)
    den = np.linalg.norm(S.reshape(len(prob.omega), -1), axis=1)
    assert (num / den).max() <= tol, num / den
    # sampled entries incl. diagonal, tile edges and the ragged tail; upper and lower triangle
    rows = np.concatenate([rng.integers(0, n_m, 40), [0, n_m - 1, 63, 64, n_m - 1, 5]])
    cols = np.concatenate([rng.integers(0, n_m, 40), [0, n_m - 1, 64, 63, 0, 5]])
    E = oracle.chi0_entries_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                                prob.omega, rows, cols, occ_tol=cfg.occ_tol)
    scale = np.abs(E).max(axis=1, keepdims=True)
    assert (np.abs(got[:, rows, cols] - E) / scale).max() <= tol


TOL_MIXED = 2e-5      # BASELINE.json:north_star, relative Frobenius error per frequency (mixed mode)


def test_cfg3_full_size_mixed():
    """cfg 3 = the metal in mixed mode, all 216 k-points, both spin channels (two contexts)."""
    cfg = get_config(3)
    prob = generate(cfg)
    for spin in range(cfg.n_spin):
        got = run_cuda(prob, spin=spin, precision=1)
        _sampled_and_sketch(prob, spin, got, TOL_MIXED)


def test_cfg3_full_size_mixed_band_batches():
    """cfg 3 spin 0, all k-points, O x U split into 16 x 32 band batches: the FP8-corrected products are
    still selected (216 * 16 * 32 >= 64 * 600) and every batch carries its own scale."""
    cfg = get_config(3)
    prob = generate(cfg)
    got = run_cuda(prob, spin=0, precision=1, max_n_o=16, max_n_u=32)
    _sampled_and_sketch(prob, 0, got, TOL_MIXED)


def test_cfg4_full_size_mixed():
    """cfg 4 in mixed mode, the launch configuration bench.py times (one batch per k-point)."""
    cfg = get_config(4)
    prob = generate(cfg)
    got = run_cuda(prob, precision=1)
    _sampled_and_sketch(prob, 0, got, TOL_MIXED)


def test_cfg4_full_size_mixed_band_batches():
    """cfg 4 in mixed mode with the O side split into 4 band batches (z workspace a quarter the size):
    every batch carries its own FP16 scale, the result must not depend on the batching."""
    cfg = get_config(4)
    prob = generate(cfg, n_k=2)
    a = run_cuda(prob, precision=1)
    b = run_cuda(prob, precision=1, max_n_o=16)
    num = np.linalg.norm((a - b).reshape(a.shape[0], -1), axis=1)
    den = np.linalg.norm(a.reshape(a.shape[0], -1), axis=1)
    assert (num / den).max() <= TOL_MIXED


def test_cfg2_full_size_fp64():
    cfg = get_config(2)
    prob = generate(cfg)
    for spin in range(cfg.n_spin):
        got = run_cuda(prob, spin=spin)
        _sampled_and_sketch(prob, spin, got, 1e-11)


def test_cfg4_full_size_fp64():
    cfg = get_config(4)
    prob = generate(cfg)
    got = run_cuda(prob)
    _sampled_and_sketch(prob, 0, got, 1e-11)


def test_wc_full_size_cfg4():
    """W^c at cfg-4 size (N_M = 2400: 38 diagonal blocks, ragged last block) from the ORACLE's chi0 of one
    k-point at three frequencies (the full-k oracle chi0 is unaffordable; the inverse does not care)."""
    import torch
    import paper_2506_03477_b200 as q
    from qsgw_synth import coulomb_eigenvalues
    cfg = get_config(4)
    prob = generate(cfg, n_k=1)
    sp = prob.spins[0]
    sel = [0, 8, 15]
    chi = oracle.hermitian_finalize_ref(oracle.chi0_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                                                        sp.f_kq, prob.omega[sel]))
    v = coulomb_eigenvalues(cfg)
    w, info = q.wc_from_chi0(torch.from_numpy(chi).cuda(), torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    got = w.cpu().numpy()
    ref = oracle.wc_ref(chi, v)
    assert int(info.item()) == 0
    num = np.linalg.norm((got - ref).reshape(len(sel), -1), axis=1)
    den = np.linalg.norm(ref.reshape(len(sel), -1), axis=1)
    assert (num / den).max() <= 1e-10, num / den
