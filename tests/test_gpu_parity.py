"""GPU parity: the CUDA path (through the C-ABI) against the oracle, element by element on the
same seeded inputs.  Tolerances (BASELINE.json:north_star): relative Frobenius error per
frequency <= 1e-11 in FP64 mode, <= 2e-5 in mixed mode."""
import dataclasses

import numpy as np
import pytest

import oracle
from qsgw_synth import WorkloadConfig, generate, get_config, scaled_config
from gpu_helpers import rel_fro_per_freq, run_cuda, sites_of

pytestmark = pytest.mark.gpu

TOL_FP64 = 1e-11
TOL_MIXED = 2e-5


def oracle_chi(prob, spin=0, n_k_norm=None):
    sp = prob.spins[spin]
    chi = oracle.chi0_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                          prob.omega, occ_tol=prob.cfg.occ_tol, n_k_norm=n_k_norm)
    return oracle.hermitian_finalize_ref(chi)


def check_hermitian(got):
    assert np.array_equal(got, np.conj(np.transpose(got, (0, 2, 1))))   # exact mirror
    assert np.all(np.diagonal(got, axis1=1, axis2=2).imag == 0.0)


@pytest.mark.parametrize("idx", [0, 1])
def test_full_config_fp64(idx):
    prob = generate(get_config(idx))
    got = run_cuda(prob)
    ref = oracle_chi(prob)
    err = rel_fro_per_freq(got, ref)
    assert err.max() <= TOL_FP64, err
    check_hermitian(got)


def test_cfg2_reduced_k_both_spins_fp64():
    cfg = get_config(2)
    prob = generate(cfg, n_k=5)
    for spin in range(cfg.n_spin):
        got = run_cuda(prob, spin=spin, n_k_norm=cfg.n_k)
        ref = oracle_chi(prob, spin=spin, n_k_norm=cfg.n_k)
        assert rel_fro_per_freq(got, ref).max() <= TOL_FP64
    # the metal really exercises the occupation filter and both signs of D
    sp = prob.spins[0]
    w = oracle.pair_weights(sp.eps_k[0], sp.f_k[0], sp.eps_kq[0], sp.f_kq[0], prob.omega)
    assert (w[0] == 0).any() and (w[0] > 0).any() and (w[0] < 0).any()


def test_cfg4_one_kpoint_full_matrix_fp64():
    """cfg 4 extents (N_M = 2400: 38 tiles with a ragged 32-column tail; 21504 pairs per k)."""
    cfg = get_config(4)
    prob = generate(cfg, n_k=1)
    got = run_cuda(prob, n_k_norm=cfg.n_k)
    sp = prob.spins[0]
    # full 2400^2 oracle for two frequencies only (bounded CPU time), all 16 on the GPU
    sel = [0, 9]
    chi = oracle.chi0_ref(sites_of(prob), sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq,
                          prob.omega[sel], n_k_norm=cfg.n_k)
    ref = oracle.hermitian_finalize_ref(chi)
    assert rel_fro_per_freq(got[sel], ref).max() <= TOL_FP64
    check_hermitian(got[:2])


RAGGED = WorkloadConfig(name="ragged", index=77, orb_per_site=(3, 7, 1, 12), pb_per_site=(5, 23, 1, 70),
                        n_k=3, n_spin=1, n_o=5, n_u=9, n_freq=5, kind="insulator",
                        eps_occ=(-0.45, 0.0), eps_unocc=(0.02, 1.1))


def test_ragged_sites_and_pair_tail():
    """Sites of unequal size (column groups straddle site boundaries), N_M = 99 (not a multiple of
    16 or 64), 45 pairs per k (not a multiple of the 16-pair stage)."""
    prob = generate(RAGGED)
    got = run_cuda(prob)
    assert rel_fro_per_freq(got, oracle_chi(prob)).max() <= TOL_FP64
    check_hermitian(got)


@pytest.mark.parametrize("mo,mu", [(2, 9), (5, 4), (1, 1), (3, 5)])
def test_band_batching_equals_single_batch(mo, mu):
    prob = generate(RAGGED)
    got = run_cuda(prob, max_n_o=mo, max_n_u=mu)
    assert rel_fro_per_freq(got, oracle_chi(prob)).max() <= TOL_FP64


@pytest.mark.parametrize("precision,tol", [(0, TOL_FP64), (1, TOL_MIXED)])
@pytest.mark.parametrize("batches", [1, 2, 7])
def test_staged_batches_per_launch(precision, tol, batches):
    """Band batches are staged back to back in the z workspace and accumulated by one stage (b) launch per
    full workspace: 1, 2 or 7 batches per launch (a flush in the middle of a k-point, a partial last flush at
    finalize) must all give the oracle's result.  cfg 1 shapes, 5 k-points, 2 x 23 band batches."""
    cfg = get_config(1)
    prob = generate(cfg, n_k=5)
    got = run_cuda(prob, precision=precision, max_n_o=2, max_n_u=23, options={"stage_batches": batches})
    assert rel_fro_per_freq(got, oracle_chi(prob)).max() <= tol


@pytest.mark.parametrize("precision,tol", [(0, TOL_FP64), (1, TOL_MIXED)])
def test_sync_between_build_and_accumulate(precision, tol):
    """A qsgw_sync (or finalize) between zmel_build and chi0_accumulate(d_z = NULL) flushes the batches staged
    below the one just built; the built batch must still be accumulated from the slot it was written to, and the
    released slots must contribute nothing.  [build, accumulate] x 2, build, sync, accumulate per k-point, with
    three batches staged per launch, against the oracle."""
    import torch
    import paper_2506_03477_b200 as q
    cfg = get_config(1)
    prob = generate(cfg, n_k=3)
    sp = prob.spins[0]
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, 3, 2, 16, precision=precision)
    ctx.set_option("stage_batches", 3)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for k in range(3):
        Ck, Ckq = t(sp.Ck[k]), t(sp.Ckq[k])
        batches = [(n0, u0) for n0 in (0, 2) for u0 in (0, 16, 32)]       # 2 x {16, 16, 14} bands
        for i, (n0, u0) in enumerate(batches):
            nu = min(16, cfg.n_u - u0)
            ctx.zmel_build(Ck, Ckq, n0, 2, u0, nu)
            if i % 3 == 2:
                ctx.sync()                                              # flushes the two batches staged below
            ctx.chi0_accumulate(t(sp.eps_k[k, n0:n0 + 2]), t(sp.f_k[k, n0:n0 + 2]), t(sp.eps_kq[k, u0:u0 + nu]),
                                t(sp.f_kq[k, u0:u0 + nu]), 2, nu)
    got = ctx.chi0_finalize().cpu().numpy()
    ctx.destroy()
    assert rel_fro_per_freq(got, oracle_chi(prob)).max() <= tol


def test_zmel_export_matches_oracle_and_import_roundtrip():
    import torch
    import paper_2506_03477_b200 as q
    prob = generate(RAGGED)
    cfg = prob.cfg
    sp = prob.spins[0]
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, cfg.n_o, cfg.n_u)
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    zs = []
    for k in range(cfg.n_k):
        z = torch.empty((cfg.n_o, cfg.n_u, cfg.n_m), dtype=torch.complex128, device="cuda")
        ctx.zmel_build(torch.from_numpy(sp.Ck[k]).cuda(), torch.from_numpy(sp.Ckq[k]).cuda(),
                       0, cfg.n_o, 0, cfg.n_u, d_z_out=z)
        zref = oracle.zmel_ref(sites_of(prob), sp.Ck[k], sp.Ckq[k])
        zg = z.cpu().numpy()
        assert np.abs(zg - zref).max() <= 1e-13 * np.abs(zref).max()
        zs.append(z)
        # sub-batch with band offsets
        z2 = torch.empty((2, 4, cfg.n_m), dtype=torch.complex128, device="cuda")
        ctx.zmel_build(torch.from_numpy(sp.Ck[k]).cuda(), torch.from_numpy(sp.Ckq[k]).cuda(),
                       3, 2, 5, 4, d_z_out=z2)
        assert np.abs(z2.cpu().numpy() - zref[3:5, 5:9]).max() <= 1e-13 * np.abs(zref).max()
    # stage (b) alone, driven with imported z (here: oracle z -> pins stage (b) independently)
    ctx.reset()
    for k in range(cfg.n_k):
        zref = torch.from_numpy(oracle.zmel_ref(sites_of(prob), sp.Ck[k], sp.Ckq[k])).cuda()
        ctx.chi0_accumulate(torch.from_numpy(sp.eps_k[k]).cuda(), torch.from_numpy(sp.f_k[k]).cuda(),
                            torch.from_numpy(sp.eps_kq[k]).cuda(), torch.from_numpy(sp.f_kq[k]).cuda(),
                            cfg.n_o, cfg.n_u, d_z=zref)
    got = ctx.chi0_finalize().cpu().numpy()
    assert rel_fro_per_freq(got, oracle_chi(prob)).max() <= TOL_FP64
    ctx.destroy()


def test_degenerate_cases():
    """N_M = 1 with one pair (scalar chi0 = w |z|^2); D = 0 at omega = 0 (dropped, reading R3);
    all pairs dropped by the occupation filter (exact zeros)."""
    import torch
    import paper_2506_03477_b200 as q
    t = lambda a, dt=np.float64: torch.from_numpy(np.asarray(a, dtype=dt)).cuda()
    ctx = q.Chi0Context([1], [1], [0.0, 0.5], 1, 1, 1)
    ctx.set_product_tensor(t([0.5 - 1.5j], np.complex128))
    Ck = t([[0.6 + 0.8j]], np.complex128); Ckq = t([[-0.28 + 0.96j]], np.complex128)
    ctx.zmel_build(Ck, Ckq, 0, 1, 0, 1)
    ctx.chi0_accumulate(t([-0.2]), t([1.0]), t([0.3]), t([0.0]), 1, 1)
    got = ctx.chi0_finalize().cpu().numpy()
    zabs2 = abs(0.5 - 1.5j) ** 2
    assert got[0, 0, 0] == pytest.approx(-2 * 0.5 / 0.25 * zabs2, rel=1e-14)
    assert got[1, 0, 0] == pytest.approx(-2 * 0.5 / 0.5 * zabs2, rel=1e-14)
    # D = 0: omega_0 = 0 gives 0/0 -> 0, omega_1 gives 0 numerator
    ctx.reset()
    ctx.zmel_build(Ck, Ckq, 0, 1, 0, 1)
    ctx.chi0_accumulate(t([0.1]), t([0.5]), t([0.1]), t([0.5]), 1, 1)
    got = ctx.chi0_finalize().cpu().numpy()
    assert np.all(got == 0.0) and np.all(np.isfinite(got))
    # occupation filter drops everything (f(1-f') = 1e-13 <= 1e-12)
    ctx.reset()
    ctx.zmel_build(Ck, Ckq, 0, 1, 0, 1)
    ctx.chi0_accumulate(t([-0.2]), t([1.0]), t([0.3]), t([1.0 - 1e-13]), 1, 1)
    assert np.all(ctx.chi0_finalize().cpu().numpy() == 0.0)
    ctx.destroy()


def test_state_machine_and_shape_errors():
    import torch
    import paper_2506_03477_b200 as q
    prob = generate(RAGGED, n_k=1)
    cfg = prob.cfg
    sp = prob.spins[0]
    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, 1, 3, 4)
    Ck = torch.from_numpy(sp.Ck[0]).cuda(); Ckq = torch.from_numpy(sp.Ckq[0]).cuda()
    e = [torch.from_numpy(x[0]).cuda() for x in (sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq)]
    with pytest.raises(q.QsgwError) as ei:
        ctx.zmel_build(Ck, Ckq, 0, 2, 0, 2)              # before set_product_tensor
    assert ei.value.code == 3
    ctx.set_product_tensor(torch.from_numpy(prob.P).cuda())
    with pytest.raises(q.QsgwError) as ei:
        ctx.chi0_accumulate(*e, 2, 2)                    # no batch built
    assert ei.value.code == 3
    with pytest.raises(q.QsgwError) as ei:
        ctx.zmel_build(Ck, Ckq, 0, 4, 0, 2)              # n_o > max_n_o
    assert ei.value.code == 2
    with pytest.raises(q.QsgwError) as ei:
        ctx.zmel_build(Ck, Ckq, 0, 0, 0, 2)              # empty batch
    assert ei.value.code == 2
    with pytest.raises(q.QsgwError) as ei:
        ctx.zmel_build(Ck, Ckq, 0, 2, 0, 2, ld_k=cfg.n_b - 1)
    assert ei.value.code == 1
    ctx.zmel_build(Ck, Ckq, 0, 2, 0, 3)
    with pytest.raises(q.QsgwError) as ei:
        ctx.chi0_accumulate(*e, 2, 2)                    # mismatched batch
    assert ei.value.code == 2
    ctx.chi0_accumulate(e[0][:2], e[1][:2], e[2][:3], e[3][:3], 2, 3)
    with pytest.raises(q.QsgwError) as ei:
        ctx.chi0_accumulate(e[0][:2], e[1][:2], e[2][:3], e[3][:3], 2, 3)   # batch already consumed
    assert ei.value.code == 3
    assert ctx.pairs_accumulated == 6 and ctx.kernel_launches >= 2     # zmel + weights; the batch is staged
    n0 = ctx.kernel_launches
    ctx.sync()                                                          # sync accumulates what is staged
    assert ctx.kernel_launches == n0 + 1
    ctx.sync()
    assert ctx.kernel_launches == n0 + 1                                # nothing staged any more
    with pytest.raises(q.QsgwError) as ei:
        q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, 1, 64, 64, workspace_bytes=1024)
    assert ei.value.code == 4
    ctx.destroy()


def test_reset_and_repeat_finalize():
    prob = generate(get_config(0), n_k=2)
    got, ctx = run_cuda(prob, return_ctx=True)
    again = ctx.chi0_finalize().cpu().numpy()
    assert np.array_equal(got, again)
    ctx.reset()
    assert np.all(ctx.chi0_finalize().cpu().numpy() == 0.0)
    ctx.destroy()


def test_run_host_entry_matches_device_path():
    import paper_2506_03477_b200 as q
    prob = generate(get_config(0), n_k=3)
    cfg = prob.cfg
    sp = prob.spins[0]
    out, launches = q.chi0_run_host(cfg.orb_per_site, cfg.pb_per_site, prob.omega, prob.P, sp.Ck, sp.Ckq,
                                    sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq, cfg.n_o, cfg.n_u)
    assert launches >= 3 * 2 + 2          # per k-point zmel + weights; staged stage (b) launch + finalize
    assert rel_fro_per_freq(out, oracle_chi(prob)).max() <= TOL_FP64


def test_invariants_on_gpu_output():
    """Properties that hold at any size: Hermitian, negative semidefinite,
    monotone decay with omega, on the CUDA result itself (cfg 1, all k)."""
    prob = generate(get_config(1))
    got = run_cuda(prob)
    nrm = np.linalg.norm(got, axis=(1, 2))
    for j in range(got.shape[0]):
        ev = np.linalg.eigvalsh(got[j])
        assert ev.max() <= 1e-12 * abs(ev.min())
    assert np.all(np.diff(nrm) < 0)


@pytest.mark.parametrize("seed", range(8))
def test_random_small_shapes(seed):
    """Seeded random cells: 1-6 sites with 1-14 orbitals and 1-40 product functions each (column groups that
    straddle up to several sites, N_M below one tile or over several), 1-7 x 1-19 bands, random band batches,
    1-6 frequencies; FP64 at 1e-11 and mixed at 2e-5 against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    s = int(rng.integers(1, 7))
    cfg = WorkloadConfig(name=f"rand{seed}", index=100 + seed,
                         orb_per_site=tuple(int(x) for x in rng.integers(1, 15, s)),
                         pb_per_site=tuple(int(x) for x in rng.integers(1, 41, s)),
                         n_k=int(rng.integers(1, 5)), n_spin=1, n_o=1, n_u=1, n_freq=int(rng.integers(1, 7)),
                         kind="insulator", eps_occ=(-0.45, 0.0), eps_unocc=(0.02, 1.1))
    if sum(cfg.orb_per_site) < 2:                                    # the generator needs two bands
        cfg = dataclasses.replace(cfg, orb_per_site=(2,) + cfg.orb_per_site[1:])
    n_b = sum(cfg.orb_per_site)
    n_o = int(rng.integers(1, min(7, n_b - 1) + 1))                 # the generator takes O and U from disjoint columns
    n_u = int(rng.integers(1, min(19, n_b - n_o) + 1))
    cfg = dataclasses.replace(cfg, n_o=n_o, n_u=n_u)
    prob = generate(cfg)
    ref = oracle_chi(prob)
    mo, mu = int(rng.integers(1, n_o + 1)), int(rng.integers(1, n_u + 1))
    for precision, tol in ((0, TOL_FP64), (1, TOL_MIXED)):
        got = run_cuda(prob, precision=precision, max_n_o=mo, max_n_u=mu)
        err = rel_fro_per_freq(got, ref).max()
        assert err <= tol, (cfg, mo, mu, precision, err)
        check_hermitian(got)


@pytest.mark.parametrize("precision,tol", [(0, TOL_FP64), (1, TOL_MIXED)])
@pytest.mark.parametrize("case", ["cfg0", "cfg1", "ragged", "cfg1_groups", "cfg1_band_batches"])
def test_add_kpoints_multi_k_launches(case, precision, tol):
    """qsgw_chi0_add_kpoints: the k-points that fit the z workspace are built by one stage (a) launch and one weight
    launch (grid.z = k-point, one FP16 scale per k-point in mixed mode).  Whole cfg 0 / cfg 1 jobs in one group, the
    ragged cell, cfg 1 forced into groups of 3 k-points (flushes between groups, a partial last group), and the
    fallback through the band-batch loop when a k-point does not fit one band batch -- all against the oracle, and
    with far fewer launches than the k-point-by-k-point path."""
    opts, kw = {}, {}
    if case == "cfg0":
        prob = generate(get_config(0))
    elif case == "ragged":
        prob = generate(RAGGED)
    else:
        prob = generate(get_config(1), n_k=20)
        if case == "cfg1_groups":
            opts = {"stage_batches": 3}
        if case == "cfg1_band_batches":
            kw = {"max_n_o": 3, "max_n_u": 20}
    n_k_norm = prob.cfg.n_k
    st, st1 = {}, {}
    got = run_cuda(prob, precision=precision, n_k_norm=n_k_norm, options=opts, stats=st, multi_k=True, **kw)
    assert rel_fro_per_freq(got, oracle_chi(prob, n_k_norm=n_k_norm)).max() <= tol
    check_hermitian(got)
    one = run_cuda(prob, precision=precision, n_k_norm=n_k_norm, options=opts, stats=st1, **kw)
    if precision == 0:
        assert rel_fro_per_freq(got, one).max() <= 1e-14          # same kernels on the same slots
    if case in ("cfg0", "cfg1", "ragged"):
        assert st["kernel_launches"] <= 7 and st1["kernel_launches"] > 2 * prob.spins[0].Ck.shape[0]


@pytest.mark.parametrize("precision,tol", [(0, TOL_FP64), (1, 2e-5)])
def test_dead_stage_skipping_forced(precision, tol):
    """Option "skip_dead_stages" = 2 (default: only large flushes): stage (b) runs only the 32-pair stages that carry weight.
    Metal-like occupations (cfg 2 shape, 3 k-points): whole bands n fail the occupation filter, so runs of stages are dead;
    then every pair dropped (no live stage at all: exact zeros); both through the multi-k launch."""
    cfg = get_config(2)
    prob = generate(cfg, n_k=3)
    sp = prob.spins[0]
    f_k = sp.f_k.copy()
    f_k[:, -4:] = 0.0                                    # the four highest O bands empty at every k: 280 consecutive dead pairs
    sp = dataclasses.replace(sp, f_k=f_k)
    prob = dataclasses.replace(prob, spins=[sp])
    keep = sp.f_k[:, :, None] * (1.0 - sp.f_kq[:, None, :]) > cfg.occ_tol
    dead = [int((~keep[k].reshape(-1)[:keep[k].size // 32 * 32].reshape(-1, 32).any(1)).sum()) for k in range(3)]
    assert min(dead) >= 7                                # the case really has dead stages
    ref = oracle_chi(prob, n_k_norm=cfg.n_k)
    for multi_k in (False, True):
        got = run_cuda(prob, precision=precision, n_k_norm=cfg.n_k, options={"skip_dead_stages": 2}, multi_k=multi_k)
        assert rel_fro_per_freq(got, ref).max() <= tol
        off = run_cuda(prob, precision=precision, n_k_norm=cfg.n_k, options={"skip_dead_stages": 0}, multi_k=multi_k)
        assert rel_fro_per_freq(off, ref).max() <= tol
    empty = dataclasses.replace(prob, spins=[dataclasses.replace(sp, f_k=np.zeros_like(sp.f_k))])
    got = run_cuda(empty, precision=precision, n_k_norm=cfg.n_k, options={"skip_dead_stages": 2}, multi_k=True)
    assert np.all(got == 0)
