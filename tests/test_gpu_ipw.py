"""GPU parity of the interstitial-plane-wave block of the matrix elements (row f4; Eqs. 4, 5, 8, PAPER.md:106-110,130;
DESIGN.md reading R21) through the C ABI (qsgw_zmel_ipw_build) against oracle.zmel_ipw_ref on the same seeded inputs,
every element.  Tolerance 1e-12 of max |z| (FP64 on both sides, contractions of up to a few hundred terms)."""
import numpy as np
import pytest

import oracle
from qsgw_synth import WorkloadConfig, generate, synthetic_ipw
from gpu_helpers import sites_of

pytestmark = pytest.mark.gpu

TOL = 1e-12


def dev(p):
    import torch
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return dict(theta=t(p.theta), g_kq=t(p.g_kq), g_k=t(p.g_k), g_ipw=t(p.g_ipw), Bk=t(p.Bk), Bkq=t(p.Bkq))


def cuda_ipw(p, L=None, theta=None, out=None, col_offset=0):
    import torch
    import paper_2506_03477_b200 as q
    d = dev(p)
    if theta is not None:
        d["theta"] = torch.from_numpy(np.ascontiguousarray(theta)).cuda()
    z = q.zmel_ipw_build(p.L if L is None else L, d["theta"], d["g_kq"], d["g_k"], d["g_ipw"], d["Bk"], d["Bkq"], out=out,
                         col_offset=col_offset)
    torch.cuda.synchronize()
    return z


@pytest.mark.parametrize("a0,n_o,n_u,n_spheres", [(6.5, 3, 5, 1), (7.5, 8, 12, 2), (12.0, 16, 40, 4)])
def test_ipw_block_parity(a0, n_o, n_u, n_spheres):
    """30 / 120 plane waves per eigenfunction, 48 / 187 IPWs (ragged 64-tiles in every GEMM extent)."""
    p = synthetic_ipw(n_o=n_o, n_u=n_u, a0=a0, n_spheres=n_spheres, seed=int(a0))
    ref = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    got = cuda_ipw(p).cpu().numpy()
    assert got.shape == ref.shape
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_ipw_box_smaller_than_the_differences():
    """Differences outside the theta box count as zero (include/qsgw.h)."""
    p = synthetic_ipw(n_o=4, n_u=6, a0=7.5, seed=2)
    Ls = np.maximum(p.L - 2, 0)
    sl = tuple(slice(int(a - b), int(a + b) + 1) for a, b in zip(p.L, Ls))
    th = np.ascontiguousarray(p.theta[sl])
    ref = oracle.zmel_ipw_ref(th, Ls, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    full = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    assert np.abs(ref - full).max() > 1e-6 * np.abs(full).max()            # the truncation matters in this case
    got = cuda_ipw(p, L=Ls, theta=th).cpu().numpy()
    assert np.abs(got - ref).max() <= TOL * np.abs(ref).max()


def test_ipw_columns_beside_the_mt_block_feed_stage_b():
    """Mixed product basis = MT product functions + IPWs: the IPW block is written into the columns behind the MT block of
    one z array (ld_z = N_MT + n_ipw) and stage (b) accumulates chi0 over all N_M columns (qsgw_chi0_accumulate with d_z);
    oracle: chi0 from the concatenated oracle z.  The context sees the IPWs as one more 'site' of the index space."""
    import torch
    import paper_2506_03477_b200 as q
    p = synthetic_ipw(n_o=5, n_u=19, a0=7.5, seed=4)
    n_ipw = len(p.g_ipw)
    cfg = WorkloadConfig(name="mt_plus_ipw", index=78, orb_per_site=(9, 15, 1), pb_per_site=(23, 41, n_ipw), n_k=1,
                         n_spin=1, n_o=5, n_u=19, n_freq=5, kind="insulator", eps_occ=(-0.45, -0.05),
                         eps_unocc=(0.05, 1.1))
    prob = generate(cfg)
    sp = prob.spins[0]
    n_mt = 23 + 41
    sites = sites_of(prob)
    z_ref = oracle.zmel_ref(sites, sp.Ck[0], sp.Ckq[0])
    z_ref[:, :, n_mt:] = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    w = oracle.pair_weights(sp.eps_k[0], sp.f_k[0], sp.eps_kq[0], sp.f_kq[0], prob.omega)
    acc = np.zeros((cfg.n_freq, cfg.n_m, cfg.n_m), dtype=np.complex128)
    oracle.chi0_accumulate_ref(acc, z_ref, w.reshape(cfg.n_freq, -1))
    chi_ref = oracle.hermitian_finalize_ref(acc / cfg.n_k)

    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, cfg.n_o, cfg.n_u)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    z = torch.empty((cfg.n_o, cfg.n_u, cfg.n_m), dtype=torch.complex128, device="cuda")
    ctx.zmel_build(torch.from_numpy(sp.Ck[0]).cuda(), torch.from_numpy(sp.Ckq[0]).cuda(), 0, cfg.n_o, 0, cfg.n_u, d_z_out=z)
    ctx.sync()
    cuda_ipw(p, out=z, col_offset=n_mt)
    zg = z.cpu().numpy()
    assert np.abs(zg - z_ref).max() <= 1e-12 * np.abs(z_ref).max()
    ctx.reset()
    ctx.chi0_accumulate(torch.from_numpy(sp.eps_k[0]).cuda(), torch.from_numpy(sp.f_k[0]).cuda(),
                        torch.from_numpy(sp.eps_kq[0]).cuda(), torch.from_numpy(sp.f_kq[0]).cuda(), cfg.n_o, cfg.n_u, d_z=z)
    got = ctx.chi0_finalize().cpu().numpy()
    ctx.destroy()
    err = max(np.linalg.norm(got[j] - chi_ref[j]) / np.linalg.norm(chi_ref[j]) for j in range(cfg.n_freq))
    assert err <= 1e-11


def test_ipw_argument_errors():
    """Error codes of the C ABI itself (called through ctypes without the binding's own checks)."""
    import ctypes as C
    import torch
    import paper_2506_03477_b200 as q
    p = synthetic_ipw(n_o=2, n_u=3, a0=6.5, seed=9)
    d = dev(p)
    n_kq, n_k, n_i = len(p.g_kq), len(p.g_k), len(p.g_ipw)
    out = torch.zeros((2, 3, n_i), dtype=torch.complex128, device="cuda")
    ptr = lambda t: C.c_void_p(t.data_ptr())

    def call(L=p.L, theta=ptr(d["theta"]), nkq=n_kq, nk=n_k, ni=n_i, ld_k=n_k, ld_kq=n_kq, ld_z=n_i, n_o=2, n_u=3):
        hl = (C.c_int32 * 3)(int(L[0]), int(L[1]), int(L[2]))
        return q.lib().qsgw_zmel_ipw_build(hl, theta, nkq, ptr(d["g_kq"]), nk, ptr(d["g_k"]), ni, ptr(d["g_ipw"]),
                                           ptr(d["Bk"]), ld_k, n_o, ptr(d["Bkq"]), ld_kq, n_u, ptr(out), ld_z, None)
    assert call(theta=None) == 1                       # QSGW_ERR_INVALID_ARG: NULL
    assert call(ld_z=n_i - 1) == 1 and call(ld_k=n_k - 1) == 1
    assert call(ni=0) == 2 and call(n_o=0) == 2        # QSGW_ERR_SHAPE
    assert call(L=[-1, 0, 0]) == 2
    assert b"negative" in q.lib().qsgw_last_create_error()
    assert call() == 0                                 # and the valid call still works
    torch.cuda.synchronize()
    ref = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw, p.Bk, p.Bkq)
    assert np.abs(out.cpu().numpy() - ref).max() <= TOL * np.abs(ref).max()


def test_ipw_block_large_chunked():
    """~560 plane waves per eigenfunction, ~565 IPWs, 64 x 336 band pairs (the cfg-4 band batch): the gathered product
    tensor exceeds the 1 GiB workspace cap, so the alpha contraction runs in chunks that accumulate in the second GEMM.
    Oracle on 8 sampled IPW columns (every band pair)."""
    p = synthetic_ipw(n_o=64, n_u=336, a0=20.0, cut_pw=3.0, cut_ipw=3.0, n_spheres=4, seed=20)
    assert 16 * len(p.g_ipw) * (len(p.g_k) + 64) * len(p.g_kq) > (1 << 30)
    got = cuda_ipw(p)
    sel = np.linspace(0, len(p.g_ipw) - 1, 8).astype(int)
    ref = oracle.zmel_ipw_ref(p.theta, p.L, p.g_kq, p.g_k, p.g_ipw[sel], p.Bk, p.Bkq)
    g = got[:, :, sel].cpu().numpy()
    assert np.abs(g - ref).max() <= TOL * np.abs(ref).max()
