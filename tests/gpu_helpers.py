"""Shared helpers of the GPU parity tests: run a generated Problem through the C-ABI."""
import numpy as np


def sites_of(prob):
    return [prob.P_site(s) for s in range(prob.cfg.n_sites)]


def run_cuda(prob, spin=0, precision=0, max_n_o=None, max_n_u=None, n_k_norm=None, return_ctx=False, options=None,
             stats=None, multi_k=False):
    import torch
    import paper_2506_03477_b200 as q
    cfg = prob.cfg
    sp = prob.spins[spin]
    n_k = sp.Ck.shape[0]
    dev = "cuda"
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega,
                        n_k if n_k_norm is None else n_k_norm,
                        max_n_o or cfg.n_o, max_n_u or cfg.n_u, precision=precision,
                        occ_tol=cfg.occ_tol)
    for key, val in (options or {}).items():
        ctx.set_option(key, val)
    ctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
    Ck = torch.from_numpy(sp.Ck).to(dev); Ckq = torch.from_numpy(sp.Ckq).to(dev)
    ek = torch.from_numpy(sp.eps_k).to(dev); fk = torch.from_numpy(sp.f_k).to(dev)
    ekq = torch.from_numpy(sp.eps_kq).to(dev); fkq = torch.from_numpy(sp.f_kq).to(dev)
    if multi_k:                       # all k-points through qsgw_chi0_add_kpoints (one stage (a) launch per group)
        ctx.chi0_add_kpoints(Ck, Ckq, ek, fk, ekq, fkq)
    else:
        for k in range(n_k):
            ctx.chi0_add_kpoint(Ck[k], Ckq[k], ek[k], fk[k], ekq[k], fkq[k])
    out = ctx.chi0_finalize()
    if stats is not None:
        stats["kernel_launches"] = ctx.kernel_launches
    ctx.sync()
    res = out.cpu().numpy()
    if stats is not None and precision == 1:
        stats["launches"], stats["launches_fp8"], stats["min_eff_pairs"] = ctx.mixed_stats()
    if return_ctx:
        return res, ctx
    ctx.destroy()
    return res


def rel_fro_per_freq(got, ref):
    num = np.linalg.norm((got - ref).reshape(got.shape[0], -1), axis=1)
    den = np.linalg.norm(ref.reshape(ref.shape[0], -1), axis=1)
    return num / den
