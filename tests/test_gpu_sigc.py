"""GPU parity of the imaginary-axis correlation self-energy I^c (Eq. 22; Alg. 2 lines 11-25, 44)
through the C ABI (qsgw_zmel_build + qsgw_sigc_imag_accumulate) against oracle.sigc_imag_ref on the same seeded
inputs, every element of the n_qp x n_qp matrix.  Tolerance: relative Frobenius error <= 1e-10 (FP64 arithmetic on
both sides; sums of up to n_all N_M^2 n_freq ~ 1e9 terms of both signs).

Roles: the intermediate states n' of q-k are the bands of the generator's "unoccupied side" arrays (Ckq, eps_kq),
the n_qp states of q are its "occupied side" arrays of k-point 0 (one q: the same C_q and eps_q for every k)."""
import numpy as np
import pytest

import oracle
from qsgw_synth import WorkloadConfig, coulomb_eigenvalues, generate, get_config, scaled_config, synthetic_wc
from gpu_helpers import sites_of

pytestmark = pytest.mark.gpu

TOL = 1e-10


def rel_fro(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def oracle_sigc(prob, wcs, n_k_norm=None, spin=0):
    sp = prob.spins[spin]
    sites = sites_of(prob)
    n_k = sp.Ck.shape[0]
    z = [oracle.zmel_ref(sites, sp.Ckq[k], sp.Ck[0]) for k in range(n_k)]
    return oracle.sigc_imag_ref(z, sp.eps_k[0], [sp.eps_kq[k] for k in range(n_k)], wcs, prob.omega, n_k_norm=n_k_norm)


def cuda_sigc(prob, wcs, precision=0, n_k_norm=None, batch_all=None, pass_z=False, spin=0, options=None):
    """I^c through the C ABI; batch_all splits the intermediate states into band batches (Alg. 2 line 10)."""
    import torch
    import paper_2506_03477_b200 as q
    cfg, sp = prob.cfg, prob.spins[spin]
    n_k = sp.Ck.shape[0]
    n_all, n_qp = cfg.n_u, cfg.n_o
    b_all = batch_all or n_all
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, n_k if n_k_norm is None else n_k_norm,
                        b_all, n_qp, precision=precision)
    for key, val in (options or {}).items():
        ctx.set_option(key, val)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    Cq = torch.from_numpy(sp.Ck[0]).cuda()
    eq = torch.from_numpy(sp.eps_k[0]).cuda()
    sig = torch.zeros((n_qp, n_qp), dtype=torch.complex128, device="cuda")
    for k in range(n_k):
        Cqk = torch.from_numpy(sp.Ckq[k]).cuda()
        eqk = torch.from_numpy(sp.eps_kq[k]).cuda()
        wc = torch.from_numpy(wcs[k]).cuda()
        for a0 in range(0, n_all, b_all):
            na = min(b_all, n_all - a0)
            if pass_z:
                z = torch.empty((na, n_qp, cfg.n_m), dtype=torch.complex128, device="cuda")
                ctx.zmel_build(Cqk, Cq, a0, na, 0, n_qp, d_z_out=z)
                ctx.sigc_imag_accumulate(eq, eqk[a0:a0 + na], wc, na, n_qp, sig, d_z=z)
            else:
                ctx.zmel_build(Cqk, Cq, a0, na, 0, n_qp)
                ctx.sigc_imag_accumulate(eq, eqk[a0:a0 + na], wc, na, n_qp, sig)
    ctx.sync()
    out = sig.cpu().numpy()
    ctx.destroy()
    return out


def test_cfg0_chain_chi0_wc_sigc():
    """cfg 0: W^c from the oracle chain chi0 -> W^c (Eqs. 14, 10, 19) feeds Eq. 22; n_all = 28, n_qp = 8, N_M = 80."""
    prob = generate(get_config(0))
    sp = prob.spins[0]
    chi = oracle.hermitian_finalize_ref(oracle.chi0_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq,
                                                        sp.f_kq, prob.omega))
    wc = oracle.wc_ref(chi, coulomb_eigenvalues(prob.cfg))
    wcs = [wc] * prob.cfg.n_k
    ref = oracle_sigc(prob, wcs)
    got = cuda_sigc(prob, wcs)
    assert rel_fro(got, ref) <= TOL
    assert np.abs(got - got.conj().T).max() > 1e-6 * np.abs(got).max()      # Eq. 22 is not Hermitian in (n, m)


RAGGED = WorkloadConfig(name="ragged_sigc", index=77, orb_per_site=(7, 12, 5), pb_per_site=(23, 41, 35), n_k=3, n_spin=1,
                        n_o=5, n_u=19, n_freq=7, kind="insulator", eps_occ=(-0.45, 0.3), eps_unocc=(-0.2, 1.1))


@pytest.mark.parametrize("pass_z", [False, True])
@pytest.mark.parametrize("batch_all", [None, 8, 1])
def test_ragged_nonhermitian_w_band_batches(batch_all, pass_z):
    """N_M = 99 (ragged 64-tiles and 16-deep contraction steps), 95 pairs (ragged M tile), unequal sites, eps_q inside
    the range of eps_{q-k} (both signs of dE), a NON-Hermitian W^c per k-point (tells W from W^T / W^H), intermediate
    states in band batches of 8 and of 1, z taken from the context or passed by the caller."""
    prob = generate(RAGGED)
    wcs = [synthetic_wc(prob.cfg.n_m, prob.omega, seed=k, hermitian=False) for k in range(prob.cfg.n_k)]
    ref = oracle_sigc(prob, wcs)
    got = cuda_sigc(prob, wcs, batch_all=batch_all, pass_z=pass_z)
    assert rel_fro(got, ref) <= TOL


def test_cfg1_shape():
    """Si-like cell: N_M = 240, n_all = 46 intermediate states, n_qp = 4, 16 frequencies, 6 of 64 k-points."""
    cfg = get_config(1)
    prob = generate(cfg, n_k=6)
    wcs = [synthetic_wc(cfg.n_m, prob.omega, seed=k % 2) for k in range(6)]
    ref = oracle_sigc(prob, wcs, n_k_norm=cfg.n_k)
    got = cuda_sigc(prob, wcs, n_k_norm=cfg.n_k)
    assert rel_fro(got, ref) <= TOL


def test_cfg2_shape_metal():
    """Heusler-like metal: N_M = 600 (9.4 tiles), n_all = 70, n_qp = 30 (2100 pairs: 32.8 M tiles), bands straddling
    E_F so that dE changes sign inside the batch; 3 of 216 k-points."""
    cfg = get_config(2)
    prob = generate(cfg, n_k=3)
    wc = synthetic_wc(cfg.n_m, prob.omega, seed=5)
    ref = oracle_sigc(prob, [wc] * 3, n_k_norm=cfg.n_k)
    got = cuda_sigc(prob, [wc] * 3, n_k_norm=cfg.n_k)
    assert rel_fro(got, ref) <= TOL


def test_degenerate_weights_zero_dE_and_empty_tail():
    """eps_q equal to some eps_{q-k,n'} exactly (dE = 0 -> weight 0, reading R17) and a single frequency mesh
    point pair (n_freq = 2): the smallest mesh the weights are defined on."""
    cfg = scaled_config(RAGGED, n_freq=2, n_k=1)
    prob = generate(cfg)
    sp = prob.spins[0]
    sp.eps_kq[0][3] = sp.eps_k[0][1]
    sp.eps_kq[0][7] = sp.eps_k[0][4]
    wcs = [synthetic_wc(cfg.n_m, prob.omega, seed=1)]
    ref = oracle_sigc(prob, wcs)
    got = cuda_sigc(prob, wcs)
    assert rel_fro(got, ref) <= TOL


@pytest.mark.parametrize("case", ["ragged", "cfg1", "cfg2"])
def test_mixed_context_tcgen05_zw(case):
    """A QSGW_PREC_MIXED context runs the frequency loop ZW^c on tcgen05 with FP16-split operands (FP32-grade products,
    FP32 sums over mu and i, the closing contraction in FP64; the two correction products in E5M2 by default, option
    "sigc_fp8" = 0: in FP16): tolerance 1e-5 relative Frobenius on I^c (the north_star mixed bar is 2e-5); option "sigc_f64" keeps the FP64 GEMM on the FP32-grade z (<= 1e-6)."""
    if case == "ragged":
        prob = generate(RAGGED)
        n_k_norm = None
        wcs = [synthetic_wc(prob.cfg.n_m, prob.omega, seed=k, hermitian=False) for k in range(prob.cfg.n_k)]
    else:
        cfg = get_config(1 if case == "cfg1" else 2)
        prob = generate(cfg, n_k=3)
        n_k_norm = cfg.n_k
        wcs = [synthetic_wc(cfg.n_m, prob.omega, seed=k) for k in range(3)]
    ref = oracle_sigc(prob, wcs, n_k_norm=n_k_norm)
    got = cuda_sigc(prob, wcs, precision=1, n_k_norm=n_k_norm)            # default: E5M2 correction products
    err = rel_fro(got, ref)
    assert 1e-12 < err <= 1e-5, err
    got3 = cuda_sigc(prob, wcs, precision=1, n_k_norm=n_k_norm, options={"sigc_fp8": 0})   # three FP16 products per term
    err3 = rel_fro(got3, ref)
    assert 1e-12 < err3 <= 1e-5, err3
    assert not np.array_equal(got, got3)
    if case == "ragged":
        got64 = cuda_sigc(prob, wcs, precision=1, n_k_norm=n_k_norm, options={"sigc_f64": 1})
        assert 1e-12 < rel_fro(got64, ref) <= 1e-6
        got_b = cuda_sigc(prob, wcs, precision=1, n_k_norm=n_k_norm, batch_all=8, pass_z=True)
        assert rel_fro(got_b, ref) <= 1e-5


def test_state_and_shape_errors():
    import torch
    import paper_2506_03477_b200 as q
    prob = generate(RAGGED)
    cfg, sp = prob.cfg, prob.spins[0]
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, 1, cfg.n_u, cfg.n_o)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    eq = torch.from_numpy(sp.eps_k[0]).cuda()
    eqk = torch.from_numpy(sp.eps_kq[0]).cuda()
    wc = torch.from_numpy(synthetic_wc(cfg.n_m, prob.omega)).cuda()
    sig = torch.zeros((cfg.n_o, cfg.n_o), dtype=torch.complex128, device="cuda")
    with pytest.raises(q.QsgwError) as e:
        ctx.sigc_imag_accumulate(eq, eqk, wc, cfg.n_u, cfg.n_o, sig)           # no z batch yet
    assert e.value.code == 3
    ctx.zmel_build(torch.from_numpy(sp.Ckq[0]).cuda(), torch.from_numpy(sp.Ck[0]).cuda(), 0, cfg.n_u, 0, cfg.n_o)
    with pytest.raises(q.QsgwError) as e:
        ctx.sigc_imag_accumulate(eq, eqk, wc, cfg.n_u - 1, cfg.n_o, sig)       # differs from the built batch
    assert e.value.code == 2
    with pytest.raises(q.QsgwError) as e:
        ctx.sigc_imag_accumulate(eq, eqk, wc, cfg.n_u + 1, cfg.n_o, sig)       # larger than declared
    assert e.value.code == 2
    with pytest.raises(q.QsgwError) as e:
        ctx.sigc_imag_accumulate(eq, eqk, None, cfg.n_u, cfg.n_o, sig)
    assert e.value.code == 1
    ctx.sigc_imag_accumulate(eq, eqk, wc, cfg.n_u, cfg.n_o, sig)               # and the valid call still works
    ctx.sync()
    assert torch.isfinite(torch.view_as_real(sig)).all() and sig.abs().max() > 0
    ctx.destroy()
