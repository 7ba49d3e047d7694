"""Out-of-bounds writes into caller buffers (compute-sanitizer is closed on this GPU pool): every output
buffer of the C ABI is carved out of a larger allocation whose guard bands hold a sentinel; after the call the bands
must be untouched and the payload fully written (no sentinel left).  Ragged sizes (N_M = 99, 95 pairs) so that every
kernel runs its edge tiles."""
import numpy as np
import pytest

from qsgw_synth import WorkloadConfig, binned_pair_weights, generate, log_bin_edges, synthetic_wc

pytestmark = pytest.mark.gpu

RAGGED = WorkloadConfig(name="ragged_guard", index=79, orb_per_site=(7, 12, 5), pb_per_site=(23, 41, 35), n_k=2, n_spin=1,
                        n_o=5, n_u=19, n_freq=7, kind="insulator", eps_occ=(-0.45, 0.0), eps_unocc=(0.03, 1.1))
GUARD = 4096
SENT = -7.25e77


def guarded(shape, dtype):
    """(raw float64 buffer, complex128 view of `shape` in its middle); GUARD complex elements of sentinel on each side."""
    import torch
    n = int(np.prod(shape))
    raw = torch.full((2 * (n + 2 * GUARD),), SENT, dtype=torch.float64, device="cuda")
    view = torch.view_as_complex(raw.view(-1, 2))[GUARD:GUARD + n].view(*shape)
    return raw, view


def check(raw, view, name):
    import torch
    g = 2 * GUARD
    assert bool((raw[:g] == SENT).all()) and bool((raw[-g:] == SENT).all()), f"{name}: guard band overwritten"
    payload = raw[g:-g]
    assert not bool((payload == SENT).any()), f"{name}: payload not fully written"
    assert bool(torch.isfinite(payload).all()), f"{name}: non-finite payload"


@pytest.mark.parametrize("precision", [0, 1])
def test_guard_bands_of_every_output(precision):
    import torch
    import paper_2506_03477_b200 as q
    prob = generate(RAGGED)
    cfg, sp = prob.cfg, prob.spins[0]
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, cfg.n_o, cfg.n_u, precision=precision)
    ctx.set_product_tensor(t(prob.P))
    # z export
    rz, z = guarded((cfg.n_o, cfg.n_u, cfg.n_m), "c")
    ctx.zmel_build(t(sp.Ck[0]), t(sp.Ckq[0]), 0, cfg.n_o, 0, cfg.n_u, d_z_out=z)
    ctx.chi0_accumulate(t(sp.eps_k[0]), t(sp.f_k[0]), t(sp.eps_kq[0]), t(sp.f_kq[0]), cfg.n_o, cfg.n_u)
    ctx.chi0_add_kpoints(t(sp.Ck[1:]), t(sp.Ckq[1:]), t(sp.eps_k[1:]), t(sp.f_k[1:]), t(sp.eps_kq[1:]), t(sp.f_kq[1:]))
    rc, chi = guarded((cfg.n_freq, cfg.n_m, cfg.n_m), "c")
    ctx.chi0_finalize(chi)
    ctx.sync()
    check(rz, z, "z export")
    check(rc, chi, "chi0")
    # I^c
    rs, sig = guarded((cfg.n_o, cfg.n_o), "c")
    sig.zero_()
    ctx2 = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, cfg.n_u, cfg.n_o, precision=precision)
    ctx2.set_product_tensor(t(prob.P))
    ctx2.zmel_build(t(sp.Ckq[0]), t(sp.Ck[0]), 0, cfg.n_u, 0, cfg.n_o)
    ctx2.sigc_imag_accumulate(t(sp.eps_k[0]), t(sp.eps_kq[0]), t(synthetic_wc(cfg.n_m, prob.omega)), cfg.n_u, cfg.n_o, sig)
    ctx2.sync()
    check(rs, sig, "sigc")
    ctx2.destroy()
    ctx.destroy()
    if precision == 0:
        # W^c, rotation, binned spectral part, Hilbert transform
        from qsgw_synth import coulomb_eigenvalues, haar_unitary
        rw, w = guarded(tuple(chi.shape), "c")
        info = torch.zeros(1, dtype=torch.int32, device="cuda")
        q.wc_from_chi0(chi.contiguous(), t(coulomb_eigenvalues(cfg)), out=w, info=info)
        rr, rot = guarded(tuple(chi.shape), "c")
        q.chi0_to_coulomb_basis(chi.contiguous(), t(haar_unitary(np.random.default_rng(1), cfg.n_m)), out=rot)
        edges = log_bin_edges(11, 1e-2, 2.0)
        ctx3 = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, edges[:-1], cfg.n_k, cfg.n_o, cfg.n_u)
        ctx3.set_product_tensor(t(prob.P))
        for k in range(cfg.n_k):
            bp, pr, ww = binned_pair_weights(sp.eps_k[k], sp.f_k[k], sp.eps_kq[k], sp.f_kq[k], edges, 0.2)
            ctx3.imchi_add_batch(t(sp.Ck[k]), t(sp.Ckq[k]), 0, cfg.n_o, 0, cfg.n_u, t(bp), t(pr), t(ww))
        ra, A = guarded((11, cfg.n_m, cfg.n_m), "c")
        ctx3.chi0_finalize(A)
        rh, h = guarded((cfg.n_freq, cfg.n_m, cfg.n_m), "c")
        q.hilbert_to_imag_axis(A, t(edges), t(prob.omega), out=h)
        ctx3.sync()
        torch.cuda.synchronize()
        assert int(info.item()) == 0
        for raw, view, name in ((rw, w, "W^c"), (rr, rot, "rotation"), (ra, A, "A (bins)"), (rh, h, "Hilbert")):
            check(raw, view, name)
        ctx3.destroy()
