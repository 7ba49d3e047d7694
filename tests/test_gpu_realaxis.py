"""GPU parity of the paper's real-axis route (Eqs. 15-18; Alg. 1 lines 9-27) through the C ABI
(qsgw_imchi_add_batch, qsgw_chi0_finalize, qsgw_hilbert_to_imag_axis) against oracle.imchi_ref / hilbert_imag_ref on
the same seeded inputs, every element.  Tolerance: relative Frobenius error per bin <= 1e-11 (FP64 sums of positive
terms, the north_star FP64 bar; empty bins must be exactly zero); Hilbert transform <= 1e-12."""
import numpy as np
import pytest

import oracle
from qsgw_synth import WorkloadConfig, binned_pair_weights, generate, get_config, log_bin_edges, scaled_config
from gpu_helpers import sites_of

pytestmark = pytest.mark.gpu


def weights_of(prob, edges, rel_width, spin=0):
    sp = prob.spins[spin]
    return [binned_pair_weights(sp.eps_k[k], sp.f_k[k], sp.eps_kq[k], sp.f_kq[k], edges, rel_width, prob.cfg.occ_tol)
            for k in range(sp.Ck.shape[0])]


def batch_csr(w, n_u, n0, no, u0, nu, n_bins):
    """The CSR triple of the band batch n in [n0, n0+no), n' in [u0, u0+nu) with batch-local pair indices."""
    bp, pr, ww = w
    n, u = pr // n_u, pr % n_u
    sel = (n >= n0) & (n < n0 + no) & (u >= u0) & (u < u0 + nu)
    bins = np.repeat(np.arange(n_bins), np.diff(bp))[sel]
    ptr = np.zeros(n_bins + 1, dtype=np.int32)
    np.add.at(ptr, bins + 1, 1)
    return np.cumsum(ptr).astype(np.int32), ((n[sel] - n0) * nu + (u[sel] - u0)).astype(np.int32), ww[sel]


def cuda_imchi(prob, edges, wts, n_k_norm=None, max_n_o=None, max_n_u=None, spin=0, stats=None, precision=0, options=None):
    import torch
    import paper_2506_03477_b200 as q
    cfg, sp = prob.cfg, prob.spins[spin]
    n_k, n_bins = sp.Ck.shape[0], len(edges) - 1
    mo, mu = max_n_o or cfg.n_o, max_n_u or cfg.n_u
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, edges[:-1], n_k if n_k_norm is None else n_k_norm, mo, mu,
                        precision=precision)
    for key, val in (options or {}).items():
        ctx.set_option(key, val)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for k in range(n_k):
        Ck, Ckq = t(sp.Ck[k]), t(sp.Ckq[k])
        for n0 in range(0, cfg.n_o, mo):
            for u0 in range(0, cfg.n_u, mu):
                no, nu = min(mo, cfg.n_o - n0), min(mu, cfg.n_u - u0)
                bp, pr, ww = batch_csr(wts[k], cfg.n_u, n0, no, u0, nu, n_bins)
                ctx.imchi_add_batch(Ck, Ckq, n0, no, u0, nu, t(bp), t(pr) if len(pr) else None, t(ww) if len(pr) else None)
    out = ctx.chi0_finalize()
    ctx.sync()
    if stats is not None:
        stats["launches"] = ctx.kernel_launches
    res = out.cpu().numpy()
    ctx.destroy()
    return res


def check_bins(got, ref, tol=1e-11):
    for j in range(ref.shape[0]):
        nr = np.linalg.norm(ref[j])
        if nr == 0.0:
            assert np.all(got[j] == 0), j
        else:
            assert np.linalg.norm(got[j] - ref[j]) / nr <= tol, (j, np.linalg.norm(got[j] - ref[j]) / nr)
    assert np.array_equal(got, np.conj(np.transpose(got, (0, 2, 1))))


@pytest.mark.parametrize("idx,n_bins", [(0, 24), (1, 100)])
def test_imchi_small_configs(idx, n_bins):
    cfg = get_config(idx)
    prob = generate(cfg, n_k=min(cfg.n_k, 12))
    edges = log_bin_edges(n_bins, 5e-3, 2.0)
    wts = weights_of(prob, edges, 0.08)
    sp = prob.spins[0]
    ref = oracle.hermitian_finalize_ref(oracle.imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, n_bins, n_k_norm=cfg.n_k))
    got = cuda_imchi(prob, edges, wts, n_k_norm=cfg.n_k)
    check_bins(got, ref)
    assert any(np.all(ref[j] == 0) for j in range(n_bins))          # the mesh really has empty bins


RAGGED = WorkloadConfig(name="ragged_bins", index=78, orb_per_site=(7, 12, 5), pb_per_site=(23, 41, 35), n_k=3, n_spin=1,
                        n_o=5, n_u=19, n_freq=7, kind="insulator", eps_occ=(-0.45, 0.0), eps_unocc=(0.03, 1.1))


@pytest.mark.parametrize("mo,mu", [(None, None), (2, 7), (1, 1)])
def test_imchi_ragged_sites_and_band_batches(mo, mu):
    """N_M = 99, 95 pairs per k-point (ragged 32-pair stages), wide windows (a pair in up to ~6 bins), band batches
    down to a single pair: every batch is sorted and accumulated on its own."""
    prob = generate(RAGGED)
    edges = log_bin_edges(30, 1e-2, 2.0)
    wts = weights_of(prob, edges, 0.3)
    sp = prob.spins[0]
    ref = oracle.hermitian_finalize_ref(oracle.imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, 30))
    got = cuda_imchi(prob, edges, wts, max_n_o=mo, max_n_u=mu)
    check_bins(got, ref)


def test_imchi_metal_cfg2_shape():
    """The metal: pairs dropped by the occupation filter and by D <= 0 carry no entry (they sort behind every bin),
    fractional occupation factors; N_M = 600, 5 of 216 k-points, 100 bins."""
    cfg = get_config(2)
    prob = generate(cfg, n_k=5)
    edges = log_bin_edges(100, 1e-3, 1.5)
    wts = weights_of(prob, edges, 0.05)
    sp = prob.spins[0]
    assert len(wts[0][1]) < cfg.n_o * cfg.n_u * 3 and len(set(wts[0][1])) < cfg.n_o * cfg.n_u
    ref = oracle.hermitian_finalize_ref(oracle.imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, 100, n_k_norm=cfg.n_k))
    got = cuda_imchi(prob, edges, wts, n_k_norm=cfg.n_k)
    check_bins(got, ref)


def test_imchi_cfg4_one_kpoint_sampled_bins():
    """cfg 4 extents (N_M = 2400, 21504 pairs, 100 bins): full 2400^2 oracle for five bins (empty, sparse, the
    fullest), the sum rule over all bins through one oracle ZGEMM."""
    cfg = get_config(4)
    prob = generate(cfg, n_k=1)
    edges = log_bin_edges(100, 1e-3, 2.5)
    wts = weights_of(prob, edges, 0.05)
    sp = prob.spins[0]
    got = cuda_imchi(prob, edges, wts, n_k_norm=cfg.n_k)
    counts = np.diff(wts[0][0])
    sel = sorted({0, int(np.argmax(counts)), int(np.nonzero(counts)[0][0]), 60, 99})
    z = oracle.zmel_ref(sites_of(prob), sp.Ck[0], sp.Ckq[0]).reshape(-1, cfg.n_m)
    bp, pr, ww = wts[0]
    for j in sel:
        Zp = z[pr[bp[j]:bp[j + 1]]]
        ref = (Zp.conj().T @ (ww[bp[j]:bp[j + 1], None] * Zp)) / cfg.n_k
        ref = oracle.hermitian_finalize_ref(ref[None])[0]
        if counts[j] == 0:
            assert np.all(got[j] == 0)
        else:
            assert np.linalg.norm(got[j] - ref) / np.linalg.norm(ref) <= 1e-11
    wsum = np.zeros(z.shape[0])
    np.add.at(wsum, pr, ww)
    tot = oracle.hermitian_finalize_ref(((z.conj().T @ (wsum[:, None] * z)) / cfg.n_k)[None])[0]
    assert np.linalg.norm(got.sum(axis=0) - tot) / np.linalg.norm(tot) <= 1e-11


def test_hilbert_transform_and_chain_to_imaginary_axis():
    """Eq. (18): the GPU transform against the oracle's on the GPU's own A (<= 1e-12), and the whole chain
    A -> chi0(i omega) against the oracle chain; with narrow windows it lands near the exact Eq. (14) chi0."""
    import torch
    import paper_2506_03477_b200 as q
    cfg = get_config(1)
    prob = generate(cfg, n_k=6)
    n_bins = 200
    edges = log_bin_edges(n_bins, 5e-3, 2.0)
    wts = weights_of(prob, edges, 1e-9)
    sp = prob.spins[0]
    A = cuda_imchi(prob, edges, wts)
    om = np.concatenate([prob.omega, [3.3, 41.0, 0.123]])             # 19 targets: two passes of 16
    got = q.hilbert_to_imag_axis(torch.from_numpy(A).cuda(), torch.from_numpy(edges).cuda(),
                                 torch.from_numpy(om).cuda()).cpu().numpy()
    ref = oracle.hilbert_imag_ref(A, edges, om)
    err = np.linalg.norm((got - ref).reshape(len(om), -1), axis=1) / np.linalg.norm(ref.reshape(len(om), -1), axis=1)
    assert err.max() <= 1e-12, err
    A_ref = oracle.hermitian_finalize_ref(oracle.imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, n_bins))
    chain = oracle.hilbert_imag_ref(A_ref, edges, om)
    err = np.linalg.norm((got - chain).reshape(len(om), -1), axis=1) / np.linalg.norm(chain.reshape(len(om), -1), axis=1)
    assert err.max() <= 1e-11, err
    # real-axis targets (bin centres and a point beyond the mesh): principal-value form of the same transform
    om_r = np.concatenate([0.5 * (edges[:-1] + edges[1:])[::9], [3.7]])
    got_r = q.hilbert_to_real_axis(torch.from_numpy(A).cuda(), torch.from_numpy(edges).cuda(),
                                   torch.from_numpy(om_r).cuda()).cpu().numpy()
    ref_r = oracle.hilbert_real_ref(A, edges, om_r)
    err = np.linalg.norm((got_r - ref_r).reshape(len(om_r), -1), axis=1) / np.linalg.norm(ref_r.reshape(len(om_r), -1), axis=1)
    assert err.max() <= 1e-12, err
    exact = oracle.hermitian_finalize_ref(oracle.chi0_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                                                          sp.f_kq, prob.omega))
    dev = np.linalg.norm((got[:16] - exact).reshape(16, -1), axis=1) / np.linalg.norm(exact.reshape(16, -1), axis=1)
    assert dev.max() < 1e-2                                           # bin-width error of the histogram, not parity


def test_realaxis_errors():
    import torch
    import paper_2506_03477_b200 as q
    prob = generate(RAGGED)
    cfg, sp = prob.cfg, prob.spins[0]
    edges = log_bin_edges(7, 1e-2, 2.0)
    bp, pr, ww = weights_of(prob, edges, 0.1)[0]
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, edges[:-1], 1, cfg.n_o, cfg.n_u)
    with pytest.raises(q.QsgwError) as e:
        ctx.imchi_add_batch(t(sp.Ck[0]), t(sp.Ckq[0]), 0, cfg.n_o, 0, cfg.n_u, t(bp), t(pr), t(ww))
    assert e.value.code == 3                                          # no product tensor yet
    ctx.set_product_tensor(t(prob.P))
    with pytest.raises(q.QsgwError) as e:
        ctx.imchi_add_batch(t(sp.Ck[0]), t(sp.Ckq[0]), 0, cfg.n_o + 1, 0, cfg.n_u, t(bp), t(pr), t(ww))
    assert e.value.code == 2
    # an empty weight list is legal and adds nothing
    ctx.imchi_add_batch(t(sp.Ck[0]), t(sp.Ckq[0]), 0, cfg.n_o, 0, cfg.n_u, t(np.zeros(8, dtype=np.int32)), None, None)
    assert float(ctx.chi0_finalize().abs().max()) == 0.0
    ctx.destroy()
    with pytest.raises(q.QsgwError):
        q.hilbert_to_imag_axis(torch.zeros((400, 4, 4), dtype=torch.complex128, device="cuda"),
                               torch.linspace(1, 2, 401, dtype=torch.float64, device="cuda"),
                               torch.zeros(1, dtype=torch.float64, device="cuda"))


@pytest.mark.parametrize("case", ["ragged", "ragged_batches", "cfg1", "cfg2"])
def test_imchi_mixed_mode(case):
    """The binned spectral part on a QSGW_PREC_MIXED context: FP16-split rows, the per-bin products on tcgen05 over the
    per-bin row ranges (three FP16 products: a bin holds too few pairs for the E5M2 corrections), the caller's weights
    scaled by the batch's 2^(-2S).  Tolerance: the north_star mixed bar, 2e-5 relative Frobenius per bin."""
    kw = {}
    if case.startswith("ragged"):
        prob, n_bins, n_k_norm = generate(RAGGED), 30, None
        edges = log_bin_edges(n_bins, 1e-2, 2.0)
        wts = weights_of(prob, edges, 0.3)
        if case == "ragged_batches":
            kw = {"max_n_o": 2, "max_n_u": 7}
    else:
        cfg = get_config(1 if case == "cfg1" else 2)
        prob, n_bins, n_k_norm = generate(cfg, n_k=5), 100, cfg.n_k
        edges = log_bin_edges(n_bins, 1e-3, 2.0)
        wts = weights_of(prob, edges, 0.06)
    sp = prob.spins[0]
    ref = oracle.hermitian_finalize_ref(oracle.imchi_ref(sites_of(prob), sp.Ck, sp.Ckq, wts, n_bins, n_k_norm=n_k_norm))
    got = cuda_imchi(prob, edges, wts, n_k_norm=n_k_norm, precision=1, **kw)
    check_bins(got, ref, tol=2e-5)
    worst = max(np.linalg.norm(got[j] - ref[j]) / np.linalg.norm(ref[j]) for j in range(n_bins) if np.linalg.norm(ref[j]) > 0)
    assert worst > 1e-12          # really the FP32-grade path
    # the same with stage (a) on tcgen05 (writes the rows through the bin sort's row map)
    got_d = cuda_imchi(prob, edges, wts, n_k_norm=n_k_norm, precision=1, options={"zmel_direct": 2}, **kw)
    check_bins(got_d, ref, tol=2e-5)
    assert not np.array_equal(got_d, got)
