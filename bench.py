#!/usr/bin/env python
"""bench.py -- chi0(q, i*omega) build throughput on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one synthetic workload: for every spin channel
and k-point {qsgw_zmel_build, qsgw_chi0_accumulate} over all band batches (driven by
qsgw_chi0_add_kpoints), then qsgw_chi0_finalize.  Default workload: cfg 4 (superlattice-scale cell),
the configuration the BASELINE.json targets are quoted on.

  value      credited complex-arithmetic TFLOP/s (8 real flop per complex multiply-add; stage (a)
             two-step count + stage (b) upper triangle over kept pairs only), inputs resident in
             HBM, CUDA events on the launching stream, max over ranks.
  e2e        same metric through qsgw_chi0_run_host: pinned HOST buffers in, HOST chi0 out.
  roofline   stage (b) kernel: credited flop per launch / mean launch time (CUDA events recorded
             by the library around each launch, inside the timed region) vs the tensor-pipe peak.
  cpu_baseline  the oracle (NumPy/BLAS, FP64) on a bounded sample of the same workload.
  accuracy   error of the TIMED outputs against the oracle (outside the timed region): full matrix where the
             oracle finishes in seconds, the exact sketch chi0 @ V (32 columns, all frequencies) otherwise.
  configs    the other BASELINE.json configurations (cfg 0-3), each with throughput and accuracy.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--mode fp64|mixed|both] [--no-configs]
  python bench.py --impl reference ...      # times the oracle on the host cores
Multi-GPU: the path does not shard in this build ("replicas only"): each rank runs
the same workload; value = units of all ranks / max-over-ranks time; no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "chi0_build_complex_tflops"
UNIT = "TFLOP/s"

# Nominal dense B200 tensor peaks (guide: B200_PROFILING.md / blackwell_cuda_programming.md) used
# only as RATIOS to the measured bf16 peak of MEASURED_PEAKS.json.
# dram__bytes_read.sum + dram__bytes_write.sum of the stage (b) kernel for ONE cfg-4 k-point (21504 pairs), from the
# `ncu --set full` captures under profiles/ (r02_*_full.md; the FP16-only variant was not captured: traffic null); a launch covers the k-points staged
# in the workspace.
NCU_DRAM_BYTES_PER_KPOINT_CFG4 = {"chi0_f64_3m_kernel": (40.162e9 + 0.771e9) / 2,          # r02 captures: two k-points per launch
                                  "chi0_f16_pair_kernel<fp8>": (12.035e9 + 0.981e9) / 2, "chi0_f16_pair_kernel": None}

NOMINAL_TF = {"bf16": 2250.0, "f16": 2250.0, "tf32": 1100.0, "f64": 40.0}


# ----------------------------------------------------------------------------- bookkeeping
def kept_pairs(cfg, prob, n_k):
    """Band pairs that pass the occupation filter f_n (1-f_n') > occ_tol (an input property)."""
    import numpy as np
    tot = 0
    for sp in prob.spins:
        occ = sp.f_k[:n_k, :, None] * (1.0 - sp.f_kq[:n_k, None, :])
        tot += int(np.count_nonzero(occ > cfg.occ_tol))
    return tot


def credited_flops(cfg, n_spin, n_k, n_freq, pairs_kept):
    """(stage a, stage b) credited real flops of the job."""
    a = 8.0 * cfg.stage_a_cmac() * n_k * n_spin
    b = 8.0 * n_freq * pairs_kept * (cfg.n_m * (cfg.n_m + 1) // 2)
    return a, b


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"bf16_burst": float(p["bf16_tflops"]), "bf16_sustained": float(p["bf16_tflops_sustained"]),
                "source": "measured"}
    return {"bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


def tensor_peak(dtype_key, sustained=True):
    pk = load_peaks()
    base = pk["bf16_sustained"] if sustained else pk["bf16_burst"]
    return base * NOMINAL_TF[dtype_key] / NOMINAL_TF["bf16"], pk["source"]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "200",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), \
        int(os.environ.get("WORLD_SIZE", "1"))


def max_over_ranks(value, world, device=None):
    """MAX of a python float over all ranks (identity at world == 1)."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ----------------------------------------------------------------------------- oracle legs
def oracle_sample(cfg, prob, seconds_hint=20.0):
    """Bounded sample of the workload for the CPU legs: (n_k_sample, freq indices)."""
    # cost model: one k-point and one frequency is one (pairs x N_M)^H (pairs x N_M) ZGEMM
    flop_kf = 8.0 * cfg.n_o * cfg.n_u * cfg.n_m * cfg.n_m
    budget = seconds_hint * 150e9            # ~150 GF/s ZGEMM on 8 cores
    n_units = max(1, int(budget / flop_kf))
    n_f = min(cfg.n_freq, n_units)
    n_k = max(1, min(cfg.n_k, n_units // n_f))
    step = max(1, cfg.n_freq // n_f)
    return n_k, list(range(0, cfg.n_freq, step))[:n_f]


def run_oracle_sample(cfg, prob, n_k_s, fsel):
    """One pass of the oracle, as it stands, over the sample.  Returns (seconds, credited flops)."""
    import numpy as np
    import oracle
    sites = [prob.P_site(s) for s in range(cfg.n_sites)]
    t0 = time.perf_counter()
    for sp in prob.spins[:1]:
        oracle.chi0_ref(sites, sp.Ck[:n_k_s], sp.Ckq[:n_k_s], sp.eps_k[:n_k_s], sp.f_k[:n_k_s],
                        sp.eps_kq[:n_k_s], sp.f_kq[:n_k_s], prob.omega[fsel], occ_tol=cfg.occ_tol,
                        n_k_norm=cfg.n_k)
    dt = time.perf_counter() - t0
    sp = prob.spins[0]
    occ = sp.f_k[:n_k_s, :, None] * (1.0 - sp.f_kq[:n_k_s, None, :])
    kept = int(np.count_nonzero(occ > cfg.occ_tol))
    fa, fb = credited_flops(cfg, 1, n_k_s, len(fsel), kept)
    return dt, fa + fb


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else len(os.sched_getaffinity(0))
    except Exception:
        return len(os.sched_getaffinity(0))


def sample_text(cfg, n_k_s, fsel):
    return (f"{cfg.name}: spin 0, {n_k_s} of {cfg.n_k} k-points x {len(fsel)} of {cfg.n_freq} frequencies, "
            f"full N_M={cfg.n_m} matrix, all {cfg.n_o}x{cfg.n_u} band pairs; credited flops as for the GPU")


# ----------------------------------------------------------------------------- accuracy of the timed outputs
def accuracy_of(cfg, prob, outs, n_k):
    """outs: {mode: [chi0 per spin (NumPy)]}.  Relative Frobenius error per frequency against the oracle, max over
    spins: the full matrix when the oracle costs < ~2e11 flop, else the exact sketch chi0 @ V."""
    import numpy as np
    import oracle
    sites = [prob.P_site(s) for s in range(cfg.n_sites)]
    full = 8.0 * cfg.n_o * cfg.n_u * float(cfg.n_m) ** 2 * cfg.n_freq * n_k * cfg.n_spin < 2e11
    res = {m: np.zeros(cfg.n_freq) for m in outs}
    t0 = time.perf_counter()
    for s, sp in enumerate(prob.spins):
        a = (sites, sp.Ck[:n_k], sp.Ckq[:n_k], sp.eps_k[:n_k], sp.f_k[:n_k], sp.eps_kq[:n_k], sp.f_kq[:n_k], prob.omega)
        if full:
            ref = oracle.hermitian_finalize_ref(oracle.chi0_ref(*a, occ_tol=cfg.occ_tol, n_k_norm=cfg.n_k))
            proj = lambda x: x
        else:
            rng = np.random.default_rng(4242 + cfg.index)
            V = (rng.standard_normal((cfg.n_m, 32)) + 1j * rng.standard_normal((cfg.n_m, 32))) / np.sqrt(2)
            ref = oracle.chi0_sketch_ref(*a, V, occ_tol=cfg.occ_tol, n_k_norm=cfg.n_k)
            proj = lambda x: x @ V
        den = np.linalg.norm(ref.reshape(cfg.n_freq, -1), axis=1)
        for m, lst in outs.items():
            num = np.linalg.norm((proj(lst[s]) - ref).reshape(cfg.n_freq, -1), axis=1)
            res[m] = np.maximum(res[m], num / np.where(den > 0, den, 1.0))
    return {m: {"max_rel_frobenius_err": float(e.max()), "per_freq": [float(x) for x in e],
                "against": ("oracle.chi0_ref, full matrix" if full else
                            "oracle.chi0_sketch_ref: chi0 @ V, 32 seeded Gaussian columns (unbiased estimator of the "
                            "Frobenius error ratio)"),
                "tolerance": 1e-11 if m == "fp64" else 2e-5, "oracle_seconds": time.perf_counter() - t0}
            for m, e in res.items()}


# ----------------------------------------------------------------------------- reference arm
def main_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from qsgw_synth import generate, get_config
    cfg = get_config(args.config)
    n_k_s, fsel = oracle_sample(cfg, None, seconds_hint=args.cpu_seconds)
    prob = generate(cfg, n_k=n_k_s)
    for _ in range(args.warmup):
        run_oracle_sample(cfg, prob, n_k_s, fsel)
    tot, flops = 0.0, 0.0
    for _ in range(args.steps):
        dt, fl = run_oracle_sample(cfg, prob, n_k_s, fsel)
        tot += dt
        flops += fl
    value = flops / tot / 1e12
    cores = blas_threads()
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": cfg.name, "mode": "oracle (NumPy/BLAS FP64) on host cores",
                                            "step": "bounded sample of the workload"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": sample_text(cfg, n_k_s, fsel)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------- CUDA arm
def run_mode(args, cfg, prob, precision, mode_name, rank, local_rank, world, light=False):
    """light: one of the small side configurations (no W^c leg, no peak probes; still step, e2e and the output)."""
    import numpy as np
    import torch
    import paper_2506_03477_b200 as q

    dev = torch.device("cuda", local_rank)
    n_spin, n_f = cfg.n_spin, cfg.n_freq
    n_k = prob.spins[0].Ck.shape[0]      # == cfg.n_k unless --n-k (profiling subset)
    pairs = kept_pairs(cfg, prob, n_k)
    fa, fb = credited_flops(cfg, n_spin, n_k, n_f, pairs)
    flops_step = fa + fb

    ctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, args.max_n_o or cfg.n_o,
                        args.max_n_u or cfg.n_u, precision=precision, occ_tol=cfg.occ_tol)
    ctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
    d_in = [[torch.from_numpy(a).to(dev) for a in (sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq)]
            for sp in prob.spins]
    out = torch.empty((n_f, cfg.n_m, cfg.n_m), dtype=torch.complex128, device=dev)

    def step():
        for s in range(n_spin):
            ctx.reset()
            ctx.chi0_add_kpoints(*d_in[s])        # all k-points: one stage (a) + weight launch per workspace group
            ctx.chi0_finalize(out)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize(dev)
    ctx.set_stage_timing(True)
    l0 = ctx.kernel_launches
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize(dev)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize(dev)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    launches = ctx.kernel_launches - l0
    stage = {nm: ctx.stage_time_ms(i) for i, nm in enumerate(("zmel", "weights", "chi0", "finalize"))}
    ctx.set_stage_timing(False)
    mixed_stats = None
    if precision == q.PREC_MIXED:        # of the last step (and spin): the counters restart at every reset
        n_l, n_l8, pe = ctx.mixed_stats()
        mixed_stats = {"stage_b_launches": n_l, "with_e5m2_corrections": n_l8, "min_effective_pairs": pe,
                       "min_effective_pairs_per_product_function": pe / cfg.n_m}
    mixed_fp8 = bool(mixed_stats and mixed_stats["with_e5m2_corrections"] > 0)
    # the timed output (last step; both spins) comes back for the accuracy check, outside the timed region
    outs_host = None
    if rank == 0 and not args.no_accuracy:
        outs_host = []
        for s in range(n_spin):
            if n_spin > 1:               # `out` holds the last spin only: rebuild this spin once, untimed
                ctx.reset()
                ctx.chi0_add_kpoints(*d_in[s])
                ctx.chi0_finalize(out)
            outs_host.append(out.cpu().numpy())
    ctx.destroy()
    # next row of the scope table, reported beside the step, not inside `value`: W^c(i omega) from
    # the chi0 just built (Eqs. 10, 19): blocked Cholesky inverse of N_omega matrices of order N_M on the GPU.
    wc = None
    sigc = None
    realaxis = None
    ipw = None
    if precision == q.PREC_FP64 and not args.no_wc and not light and rank == 0:
        from qsgw_synth import coulomb_eigenvalues, haar_unitary
        import numpy as _np
        d_v = torch.from_numpy(coulomb_eigenvalues(cfg)).to(dev)
        d_U = torch.from_numpy(haar_unitary(_np.random.default_rng(7), cfg.n_m)).to(dev)   # host work before any timing
        w_out = torch.empty_like(out)
        info = torch.zeros(1, dtype=torch.int32, device=dev)
        reps = 5

        def timed(fn):
            for _ in range(3):                                    # warm-up: the GPU idled during the host-side set-up
                fn()
            ts = []
            for _ in range(reps):                                 # every repetition timed on its own; median
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                fn()
                e1.record()
                torch.cuda.synchronize(dev)
                ts.append(e0.elapsed_time(e1))
            return statistics.median(ts)

        wc_ms = timed(lambda: q.wc_from_chi0(out, d_v, out=w_out, info=info))
        wc_flop = 4.0 * n_f * float(cfg.n_m) ** 3       # n^3/2 complex multiply-adds per frequency, 8 real flop each
        wc = {"ms": wc_ms, "value": wc_flop / (wc_ms * 1e-3) / 1e12, "unit": UNIT, "info": int(info.item()),
              "credited_flop": wc_flop, "what": "qsgw_wc_from_chi0 on the FP64 chi0 of this run (spin 0 / last spin), "
              "credited n^3/6 (Cholesky) + n^3/6 (triangular inverse) + n^3/6 (X^H X) complex multiply-adds per frequency"}
        # chi0 in the Coulomb eigenbasis (U^H chi0 U; the representation Eqs. 10/19 are stated in)
        rot_ms = timed(lambda: q.chi0_to_coulomb_basis(out, d_U, out=w_out))
        wc["rotate_ms"] = rot_ms
        wc["rotate_value"] = 2 * 8.0 * n_f * float(cfg.n_m) ** 3 / (rot_ms * 1e-3) / 1e12   # two n^3 GEMMs per frequency
        # next row f2: imaginary-axis correlation self-energy I^c (Eq. 22, Alg. 2) with the W^c just computed:
        # n_qp = the O-side bands of k-point 0 (the q states), intermediate states = the U-side bands of each k-point
        if not args.no_sigc:
            q.wc_from_chi0(out, d_v, out=w_out, info=info)
            sp0 = prob.spins[0]
            n_all, n_qp, nks = cfg.n_u, cfg.n_o, min(2, n_k)
            sctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, n_all, n_qp,
                                 precision=q.PREC_FP64)
            sctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
            d_Cq = torch.from_numpy(sp0.Ck[0]).to(dev)
            d_eq = torch.from_numpy(sp0.eps_k[0]).to(dev)
            d_Cqk = torch.from_numpy(sp0.Ckq[:nks]).to(dev)
            d_eqk = torch.from_numpy(sp0.eps_kq[:nks]).to(dev)
            sig = torch.zeros((n_qp, n_qp), dtype=torch.complex128, device=dev)

            def sigc_pass(n_sub=None):
                sig.zero_()
                na = n_sub or n_all
                for k in range(nks):
                    sctx.zmel_build(d_Cqk[k], d_Cq, 0, na, 0, n_qp)
                    sctx.sigc_imag_accumulate(d_eq, d_eqk[k][:na], w_out, na, n_qp, sig)

            sigc_pass()                                            # allocates the I^c workspace
            torch.cuda.synchronize(dev)
            l_s = sctx.kernel_launches
            ts = []
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                sigc_pass()
                e1.record()
                torch.cuda.synchronize(dev)
                ts.append(e0.elapsed_time(e1))
            s_ms = statistics.median(ts)
            s_launch = (sctx.kernel_launches - l_s) // 3
            fl_a = 8.0 * nks * sum(m * b * n_all * (b + n_qp) for b, m in zip(cfg.orb_per_site, cfg.pb_per_site))
            fl_zw = 8.0 * nks * n_qp * n_all * float(cfg.n_m) ** 2 * n_f
            fl_c = 8.0 * nks * n_qp * n_qp * n_all * float(cfg.n_m)
            sigc = {"ms": s_ms, "ms_runs": [round(t, 2) for t in ts], "value": (fl_a + fl_zw + fl_c) / (s_ms * 1e-3) / 1e12,
                    "unit": UNIT, "k_points": nks, "n_all": n_all, "n_qp": n_qp, "gpu_launches": s_launch,
                    "credited_flop": fl_a + fl_zw + fl_c,
                    "what": "qsgw_zmel_build + qsgw_sigc_imag_accumulate per k-point with the W^c of this run; credited "
                            "n_qp n_all N_M^2 n_omega (Table 1, I^c) + n_qp^2 n_all N_M (closing GEMM) + stage (a) "
                            "complex multiply-adds, 8 real flop each"}
            if not args.no_accuracy:
                # accuracy of this path against the oracle on the first 8 intermediate states (bounded CPU time)
                import oracle
                n_sub = min(8, n_all)
                sigc_pass(n_sub)
                torch.cuda.synchronize(dev)
                got = sig.cpu().numpy()
                wc_h = w_out.cpu().numpy()
                sites = [prob.P_site(s_) for s_ in range(cfg.n_sites)]
                zs = [oracle.zmel_ref(sites, sp0.Ckq[k][:n_sub], sp0.Ck[0]) for k in range(nks)]
                ref = oracle.sigc_imag_ref(zs, sp0.eps_k[0], [sp0.eps_kq[k][:n_sub] for k in range(nks)], [wc_h] * nks,
                                           prob.omega, n_k_norm=cfg.n_k)
                sigc["accuracy"] = {"rel_frobenius_err": float(_np.linalg.norm(got - ref) / _np.linalg.norm(ref)),
                                    "against": f"oracle.sigc_imag_ref on the first {n_sub} intermediate states of "
                                               f"{nks} k-points, W^c from the GPU", "tolerance": 1e-10}
            sig64 = None
            if not args.no_accuracy:
                sigc_pass()
                torch.cuda.synchronize(dev)
                sig64 = sig.clone()
            sctx.destroy()
            # the same pass on a QSGW_PREC_MIXED context: ZW^c on tcgen05 with FP16-split operands (sigc_f16_kernel)
            sctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, n_all, n_qp, precision=q.PREC_MIXED)
            sctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
            sigc_pass()
            torch.cuda.synchronize(dev)
            ts = []
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                sigc_pass()
                e1.record()
                torch.cuda.synchronize(dev)
                ts.append(e0.elapsed_time(e1))
            m_ms = statistics.median(ts)
            tf32_peak, psrc = tensor_peak("tf32", True)
            sigc["mixed"] = {"ms": m_ms, "ms_runs": [round(t, 2) for t in ts], "value": (fl_a + fl_zw + fl_c) / (m_ms * 1e-3) / 1e12,
                             "unit": UNIT, "peak": tf32_peak, "frac": (fl_a + fl_zw + fl_c) / (m_ms * 1e-3) / 1e12 / tf32_peak,
                             "peak_source": f"{psrc} bf16 cuBLAS sustained x nominal tf32/bf16 ratio (1100/2250)",
                             "what": "same pass on a QSGW_PREC_MIXED context: FP16 main product + two E5M2 correction products per term on "
                                     "tcgen05 (sigc_f16_kernel<fp8>), FP32 sums, closing contraction in FP64; same credited flop"}
            if sig64 is not None:
                sigc["mixed"]["rel_frobenius_dev_from_fp64"] = float((sig - sig64).norm() / sig64.norm())
                sigc["mixed"]["tolerance"] = 1e-5
            sctx.destroy()
            del d_Cq, d_Cqk, sig
        # next row f3: the paper's own real-axis route (Eqs. 15-18, Alg. 1 lines 12-27): binned spectral part of two
        # k-points with 100 logarithmic bins (seeded stand-in for the tetrahedron weights), then the Hilbert transform
        # of the 100 bin matrices to the n_freq imaginary frequencies
        if not args.no_realaxis:
            from qsgw_synth import binned_pair_weights, log_bin_edges
            del w_out
            torch.cuda.empty_cache()
            n_bins, nks = 100, min(2, n_k)
            edges = log_bin_edges(n_bins, 1e-3, 2.5)
            sp0 = prob.spins[0]
            wts = [binned_pair_weights(sp0.eps_k[k], sp0.f_k[k], sp0.eps_kq[k], sp0.f_kq[k], edges, 0.05, cfg.occ_tol)
                   for k in range(nks)]
            d_w = [[torch.from_numpy(a).to(dev) for a in w] for w in wts]
            rctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, edges[:-1], cfg.n_k, cfg.n_o, cfg.n_u, precision=q.PREC_FP64)
            rctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
            Ck, Ckq = d_in[0][0], d_in[0][1]
            A = torch.empty((n_bins, cfg.n_m, cfg.n_m), dtype=torch.complex128, device=dev)
            d_edges, d_om = torch.from_numpy(edges).to(dev), torch.from_numpy(prob.omega).to(dev)

            def ra_pass():
                rctx.reset()
                for k in range(nks):
                    rctx.imchi_add_batch(Ck[k], Ckq[k], 0, cfg.n_o, 0, cfg.n_u, *d_w[k])
                rctx.chi0_finalize(A)

            ra_ms = timed(ra_pass)
            h_out = torch.empty_like(out)
            hil_ms = timed(lambda: q.hilbert_to_imag_axis(A, d_edges, d_om, out=h_out))
            nnz = sum(len(w[1]) for w in wts)
            fl_ra = 8.0 * nnz * (cfg.n_m * (cfg.n_m + 1) // 2) + 8.0 * nks * cfg.stage_a_cmac()
            hil_bytes = 16.0 * (n_bins + n_f) * float(cfg.n_m) ** 2
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f_:
                hbm = float(json.load(f_).get("hbm_gbs", 0.0)) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else 0.0
            realaxis = {"imchi_ms": ra_ms, "imchi_value": fl_ra / (ra_ms * 1e-3) / 1e12, "unit": UNIT, "k_points": nks,
                        "n_bins": n_bins, "entries": nnz, "pairs": nks * cfg.n_o * cfg.n_u, "credited_flop": fl_ra,
                        "what": "qsgw_imchi_add_batch per k-point (sort, stage (a), per-bin products) + finalize; credited "
                                "8 x entries x N_M (N_M + 1) / 2 + stage (a)",
                        "hilbert_ms": hil_ms, "hilbert_gbs": hil_bytes / (hil_ms * 1e-3) / 1e9,
                        "hilbert_roofline": {"bound": "hbm", "achieved": hil_bytes / (hil_ms * 1e-3) / 1e9, "peak": hbm or None,
                                             "unit": "GB/s", "frac": (hil_bytes / (hil_ms * 1e-3) / 1e9 / hbm) if hbm else None,
                                             "algorithmic_bytes": hil_bytes,
                                             "what": "qsgw_hilbert_to_imag_axis: (n_bins + n_freq) N_M^2 complex128 read + written once"}}
            if not args.no_accuracy:
                import oracle
                got = h_out.cpu().numpy()
                A_h = A.cpu().numpy()
                ref = oracle.hilbert_imag_ref(A_h, edges, prob.omega)
                realaxis["hilbert_accuracy"] = float((_np.linalg.norm((got - ref).reshape(n_f, -1), axis=1) /
                                                      _np.linalg.norm(ref.reshape(n_f, -1), axis=1)).max())
                # one bin of the timed A against the oracle's gather / scale / GEMM (the fullest bin of k-point 0 + 1)
                sites = [prob.P_site(s_) for s_ in range(cfg.n_sites)]
                jb = int(_np.argmax(_np.diff(wts[0][0])))
                ref_b = _np.zeros((cfg.n_m, cfg.n_m), dtype=_np.complex128)
                for k in range(nks):
                    z = oracle.zmel_ref(sites, sp0.Ck[k], sp0.Ckq[k]).reshape(-1, cfg.n_m)
                    bp, pr, ww = wts[k]
                    Zp = z[pr[bp[jb]:bp[jb + 1]]]
                    ref_b += Zp.conj().T @ (ww[bp[jb]:bp[jb + 1], None] * Zp)
                ref_b = oracle.hermitian_finalize_ref((ref_b / cfg.n_k)[None])[0]
                realaxis["imchi_accuracy"] = {"bin": jb, "rel_frobenius_err": float(_np.linalg.norm(A_h[jb] - ref_b) / _np.linalg.norm(ref_b)),
                                              "tolerance": 1e-11}
                del A_h, got
            rctx.destroy()
            # the same binned accumulation on a QSGW_PREC_MIXED context (per-bin products on tcgen05, FP16-split rows)
            A64 = A.clone() if not args.no_accuracy else None
            rctx = q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, edges[:-1], cfg.n_k, cfg.n_o, cfg.n_u, precision=q.PREC_MIXED)
            rctx.set_product_tensor(torch.from_numpy(prob.P).to(dev))
            ram_ms = timed(ra_pass)
            realaxis["mixed"] = {"imchi_ms": ram_ms, "imchi_value": fl_ra / (ram_ms * 1e-3) / 1e12, "unit": UNIT,
                                 "what": "same pass on a QSGW_PREC_MIXED context: chi0_f16_kernel over the per-bin row ranges"}
            if A64 is not None:
                num = (A - A64).flatten(1).norm(dim=1)
                den = A64.flatten(1).norm(dim=1)
                realaxis["mixed"]["max_rel_frobenius_dev_from_fp64_per_bin"] = float((num / den.clamp_min(1e-300))[den > 0].max())
                realaxis["mixed"]["tolerance"] = 2e-5
                del A64
            rctx.destroy()
            del A, h_out
        else:
            del w_out
        del d_v, d_U
        # next row f4: the interstitial-plane-wave block of the matrix elements (Eqs. 4, 5, 8) for the band counts of this
        # configuration and a cell with ~290 plane waves per eigenfunction and ~370 IPWs (3 Ry / 3.5 Ry cutoffs)
        if not args.no_ipw:
            from qsgw_synth import synthetic_ipw
            torch.cuda.empty_cache()
            ip = synthetic_ipw(n_o=cfg.n_o, n_u=cfg.n_u, a0=16.0, cut_pw=3.0, cut_ipw=3.5, n_spheres=4, seed=1)
            t_ = lambda a: torch.from_numpy(_np.ascontiguousarray(a)).to(dev)
            di = [t_(ip.theta), t_(ip.g_kq), t_(ip.g_k), t_(ip.g_ipw), t_(ip.Bk), t_(ip.Bkq)]
            zi = torch.empty((cfg.n_o, cfg.n_u, len(ip.g_ipw)), dtype=torch.complex128, device=dev)
            ipw_ms = timed(lambda: q.zmel_ipw_build(ip.L, *di, out=zi))
            n_kq_, n_k_, n_i_ = len(ip.g_kq), len(ip.g_k), len(ip.g_ipw)
            fl_ipw = 8.0 * n_i_ * n_kq_ * cfg.n_o * (n_k_ + cfg.n_u)
            ipw = {"ms": ipw_ms, "value": fl_ipw / (ipw_ms * 1e-3) / 1e12, "unit": UNIT, "n_pw": [n_kq_, n_k_], "n_ipw": n_i_,
                   "n_o": cfg.n_o, "n_u": cfg.n_u, "credited_flop": fl_ipw,
                   "what": "qsgw_zmel_ipw_build: gather of theta differences + two FP64 tensor-pipe GEMMs; credited "
                           "n_ipw N_kq n_o (N_k + n_u) complex multiply-adds, 8 real flop each"}
            if not args.no_accuracy:
                import oracle
                sel = _np.linspace(0, n_i_ - 1, 6).astype(int)
                ref = oracle.zmel_ipw_ref(ip.theta, ip.L, ip.g_kq, ip.g_k, ip.g_ipw[sel], ip.Bk, ip.Bkq)
                got = zi[:, :, torch.from_numpy(sel).to(dev)].cpu().numpy()
                ipw["accuracy"] = {"max_abs_err_over_max": float(_np.abs(got - ref).max() / _np.abs(ref).max()),
                                   "against": "oracle.zmel_ipw_ref on 6 of the IPW columns, all band pairs", "tolerance": 1e-12}
            del di, zi
            # row f4: the generalized eigenproblem (v - v_mu O) z = 0 that yields the orthonormal basis E_mu and v_mu
            # (PAPER.md:116-118), on a seeded pencil of order N_M with a known spectrum
            from qsgw_synth import synthetic_mpb_matrices
            v_m, O_m, lam_m = synthetic_mpb_matrices(cfg.n_m, seed=1)
            d_vm, d_Om = torch.from_numpy(v_m).to(dev), torch.from_numpy(O_m).to(dev)
            q.coulomb_eigenbasis(d_vm, d_Om)                                  # warm-up (workspace pool)
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            w_g, U_g, sweeps = q.coulomb_eigenbasis(d_vm, d_Om)
            torch.cuda.synchronize(dev)
            eig_s = time.perf_counter() - t0
            Nn = (cfg.n_m + 63) // 64 * 64
            npr, rounds = Nn // 64, Nn // 32 - 1
            upd_flop = 8.0 * 64 ** 3 * (npr * (npr + 1) + npr * npr) * rounds * sweeps   # 2 GEMMs per upper tile of C, 1 per tile of Q
            ipw["eigenbasis"] = {"seconds": eig_s, "n_m": cfg.n_m, "sweeps": sweeps, "block_rounds": rounds * sweeps,
                                 "update_flop": upd_flop, "update_tflops_over_whole_call": upd_flop / eig_s / 1e12,
                                 "what": "qsgw_coulomb_eigenbasis (host-synchronised once per sweep; wall clock of the call): "
                                         "Cholesky reduction + two-sided block Jacobi (64 x 64 subproblems in shared memory, "
                                         "unitaries applied by 64^3 complex GEMMs on the FP64 tensor pipe) + back transformation; "
                                         "update_flop = the GEMM work of the block rounds, 8 real flop per complex multiply-add"}
            if not args.no_accuracy:
                import oracle
                t0 = time.perf_counter()
                w_r, U_r = oracle.coulomb_eigenbasis_ref(v_m, O_m)
                ipw["eigenbasis"]["oracle_seconds"] = time.perf_counter() - t0
                Un = U_g.cpu().numpy()
                wn = w_g.cpu().numpy()
                ipw["eigenbasis"]["accuracy"] = {
                    "eigenvalues_max_err_over_max": float(_np.abs(wn - w_r).max() / w_r.max()),
                    "residual_rel": float(_np.linalg.norm(v_m @ Un - (O_m @ Un) * wn[None, :]) / _np.linalg.norm(v_m)),
                    "orthonormality_max_dev": float(_np.abs(Un.conj().T @ O_m @ Un - _np.eye(cfg.n_m)).max()),
                    "against": "oracle.coulomb_eigenbasis_ref (LAPACK zhegvd on the host cores)", "tolerance": 1e-11}
            del d_vm, d_Om
    del d_in, out
    torch.cuda.empty_cache()

    value = world * args.steps * flops_step / (ms_total * 1e-3) / 1e12
    chi_ms, chi_n = stage["chi0"]
    # stage (b) kernel: credited flop per launch (one k-point and band batch, all frequencies)
    ach = (fb * args.steps / max(chi_n, 1)) / (chi_ms / max(chi_n, 1) * 1e-3) / 1e12 if chi_n else None
    dkey = {q.PREC_FP64: "f64", q.PREC_MIXED: "f16"}[precision]
    burst_peak, src = tensor_peak(dkey, sustained=False)
    sust_peak, _ = tensor_peak(dkey, sustained=True)
    probe = None
    if not light:
        try:      # the pipe's own issue-rate peak, measured on this device in this run
            probe, _ = q.probe_peak({"f64": q.PEAK_FP64_MMA, "f16": q.PEAK_F16_MMA}[dkey])
        except q.QsgwError:
            probe = None
    ratio_txt = f"x nominal {dkey}/bf16 ratio ({NOMINAL_TF[dkey]:g}/{NOMINAL_TF['bf16']:g})"
    if dkey == "f64":
        # MEASURED_PEAKS.json has no FP64 figure and the bf16-derived one is power-capped while FP64 is not
        # (the kernel exceeds it): the denominator is the DMMA pipe's issue rate, 64 FP64 FMA/clk/SM x SMs x
        # max SM clock, which the register-resident probe reproduces when it is not throttled.
        props = torch.cuda.get_device_properties(dev)
        derived = 2.0 * 64.0 * props.multi_processor_count * props.clock_rate * 1e3 / 1e12
        peak = max(derived, probe or 0.0)
        peak_src = (f"DMMA issue rate: 64 FP64 FMA/clk/SM x {props.multi_processor_count} SMs x "
                    f"{props.clock_rate / 1e3:.0f} MHz (qsgw_probe_peak(f64) measured {probe and round(probe, 2)} in this run)")
    else:
        # tcgen05 kernels run power-capped inside a seconds-long step: MEASURED_PEAKS.json sustained figure
        peak = sust_peak
        peak_src = f"{src} bf16 cuBLAS sustained (MEASURED_PEAKS.json) {ratio_txt}"
    # tensor-pipe flops the kernel executes per credited flop (full tiles, no padding counted): the FP64 kernel's
    # 3M product executes 3 real products per complex one (0.75 of the credited 4); the FP16 split 3 per term
    passes = {q.PREC_FP64: 0.75, q.PREC_MIXED: 3}[precision]
    kname = {"f64": "chi0_f64_3m_kernel", "f16": "chi0_f16_pair_kernel"}[dkey]
    pipe_txt = dkey
    extra = {}
    if precision == q.PREC_MIXED:
        # north_star's denominator for the mixed mode: the FP32/TF32 tensor peak = measured bf16 sustained x the
        # nominal tf32/bf16 ratio ("of measured, nominal ratio").  Beside it the pipe-time view of what runs:
        # three f16 products per term, or (E5M2 variant) one f16 + two e5m2 products = 1/P_f16 + 2/P_fp8 =
        # 2/P_f16 of pipe time per credited flop (fp8 nominal = 2 x f16).
        tf32_peak, _ = tensor_peak("tf32", True)
        pipe_peak = sust_peak / (2.0 if mixed_fp8 else 3.0)
        extra = {"peak_pipe_mix": pipe_peak, "frac_pipe_mix": (ach / pipe_peak) if ach else None,
                 "peak_pipe_mix_source": f"{src} bf16 sustained / " + ("2 (f16 main + 2 e5m2 corrections; fp8 nominal "
                                         "= 2 x f16)" if mixed_fp8 else "3 (three f16 products per term)")}
        peak = tf32_peak
        peak_src = f"{src} bf16 cuBLAS sustained (MEASURED_PEAKS.json) x nominal tf32/bf16 ratio (1100/2250)"
        if mixed_fp8:
            kname, pipe_txt = "chi0_f16_pair_kernel<fp8>", "f16 + e5m2"
        roof_exec_frac = extra["frac_pipe_mix"]
    else:
        roof_exec_frac = (ach * passes / peak) if ach else None
    roofline = {"bound": "tensor", "kernel": kname, "tensor_pipe": pipe_txt,
                "tensor_products_per_term": passes,
                "achieved_executed": (ach * passes) if ach else None,
                "frac_executed": roof_exec_frac,
                "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": (ach / peak) if ach else None,
                "traffic": (NCU_DRAM_BYTES_PER_KPOINT_CFG4[kname] * n_k * n_spin * args.steps / max(chi_n, 1)
                            if (cfg.index == 4 and NCU_DRAM_BYTES_PER_KPOINT_CFG4.get(kname) and chi_n) else None),
                "note": ("credited flops count 4 real products per complex multiply-add; the 3M kernel executes 3, so "
                         "`frac` (credited / peak) can exceed 1 while `frac_executed` stays below it"
                         if dkey == "f64" else "frac = credited / TF32 peak (north_star denominator); frac_executed = "
                         "tensor-pipe time fraction of the product mix that ran (peak_pipe_mix)"),
                **extra,
                "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum per cfg-4 k-point (profiles/) x "
                                  "k-points staged per launch; bytes",
                "peak_source": peak_src,
                "peak_probe": probe, "frac_executed_of_probe": (ach * passes / probe) if (ach and probe) else None,
                "peak_burst": burst_peak, "peak_burst_source": f"{src} bf16 burst {ratio_txt}",
                "avg_launch_ms": chi_ms / max(chi_n, 1), "launches_timed": chi_n,
                "stage_ms_per_step": {nm: v[0] / args.steps for nm, v in stage.items()}}

    # end to end through the host-buffer entry point (pinned host memory in and out)
    e2e = None
    if not args.no_e2e:
        hp = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        h_P = hp(prob.P)
        h_in = [[hp(a) for a in (sp.Ck, sp.Ckq, sp.eps_k, sp.f_k, sp.eps_kq, sp.f_kq)] for sp in prob.spins]
        h_out = torch.empty((n_f, cfg.n_m, cfg.n_m), dtype=torch.complex128).pin_memory().numpy()
        h2d = n_spin * h_P.nbytes + sum(a.nbytes for sp in h_in for a in sp)
        d2h = n_spin * h_out.nbytes

        # one context per spin, created (and its staging buffers allocated by a first call) before the clock starts
        e_ctx = [q.Chi0Context(cfg.orb_per_site, cfg.pb_per_site, prob.omega, cfg.n_k, args.max_n_o or cfg.n_o,
                               args.max_n_u or cfg.n_u, precision=precision, occ_tol=cfg.occ_tol)
                 for _ in range(n_spin)]

        def e2e_step():
            n = 0
            for s in range(n_spin):
                _, ln = e_ctx[s].run_host(h_P, *h_in[s], out=h_out)
                n += ln
            return n
        for _ in range(2):
            e2e_step()
        barrier()
        n_e = max(1, min(args.steps, args.e2e_steps))
        # every step is timed on its own: wall clock around the synchronous C-ABI call, max over ranks
        step_s = []
        for _ in range(n_e):
            t0 = time.perf_counter()
            e2e_step()
            step_s.append(max_over_ranks(time.perf_counter() - t0, world, dev))
        barrier()
        for c in e_ctx:
            c.destroy()
        dt = statistics.median(step_s)
        e2e = {"value": world * flops_step / dt / 1e12, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": 1e3 * dt, "steps": n_e,
               "ms_steps": [round(1e3 * t, 2) for t in step_s], "ms_min": 1e3 * min(step_s), "ms_max": 1e3 * max(step_s),
               "statistic": "median of the timed steps",
               "api": "qsgw_chi0_run_host on a persistent context (pinned host buffers; reset + H2D + all kernels + "
                      "D2H inside the timed region)"}

    return {"mode": mode_name, "value": value, "ms_per_step": ms_total / args.steps, "launches": launches,
            "roofline": roofline, "e2e": e2e, "clocks": clocks, "flops_step": flops_step,
            "flops_stage_a": fa, "flops_stage_b": fb, "pairs_kept": pairs, "wc": wc, "sigc": sigc, "realaxis": realaxis, "ipw": ipw, "mixed_selection": mixed_stats,
            "_out": outs_host}


def main_cuda(args):
    rank, local_rank, world = dist_env()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_2506_03477_b200 as q
    from paper_2506_03477_b200 import build as qbuild
    if rank == 0:
        qbuild.build()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    q.lib()
    from qsgw_synth import generate, get_config
    cfg = get_config(args.config)
    prob = generate(cfg, n_k=args.n_k or None)

    modes = {"fp64": [("fp64", q.PREC_FP64)], "mixed": [("mixed", q.PREC_MIXED)],
             "both": [("fp64", q.PREC_FP64), ("mixed", q.PREC_MIXED)]}[args.mode]
    if args.mode == "both" and cfg.precision == "mixed":
        modes = modes[::-1]
    res = [run_mode(args, cfg, prob, prec, name, rank, local_rank, world) for name, prec in modes]

    # the other BASELINE.json configurations, each in the mode(s) it names: throughput, e2e and accuracy
    side = []
    if not args.no_configs and not args.n_k and world == 1:
        for idx in [i for i in (0, 1, 2, 3) if i != cfg.index]:
            c2 = get_config(idx)
            p2 = generate(c2)
            m2 = [("mixed", q.PREC_MIXED)] if c2.precision == "mixed" else [("fp64", q.PREC_FP64)]
            if idx in (0, 1):
                m2 = [("fp64", q.PREC_FP64), ("mixed", q.PREC_MIXED)]
            a2 = argparse.Namespace(**{**vars(args), "max_n_o": 0, "max_n_u": 0, "steps": max(args.steps, 5),
                                       "e2e_steps": 3})
            rs = [run_mode(a2, c2, p2, prec, name, rank, local_rank, world, light=True) for name, prec in m2]
            acc = {} if args.no_accuracy else accuracy_of(c2, p2, {r["mode"]: r["_out"] for r in rs}, c2.n_k)
            side.append({"workload": c2.name, "n_m": c2.n_m, "n_k": c2.n_k, "n_spin": c2.n_spin,
                         "modes": [{"mode": r["mode"], "value": r["value"], "unit": UNIT, "ms_per_step": r["ms_per_step"],
                                    "gpu_launches": r["launches"], "credited_flop_per_step": r["flops_step"],
                                    "stage_b_kernel_tflops": r["roofline"]["achieved"],
                                    "stage_ms_per_step": r["roofline"]["stage_ms_per_step"],
                                    "e2e": r["e2e"] and {k: r["e2e"][k] for k in ("value", "ms_per_step", "ms_min", "ms_max")},
                                    "mixed_selection": r["mixed_selection"], "accuracy": acc.get(r["mode"])}
                                   for r in rs]})
            del p2, rs
    if rank != 0:
        return 0
    if not args.no_accuracy:
        acc = accuracy_of(cfg, prob, {r["mode"]: r["_out"] for r in res}, prob.spins[0].Ck.shape[0])
        for r in res:
            r["accuracy"] = acc[r["mode"]]
    for r in res:
        r.pop("_out", None)
    main = res[0]
    line = {"metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp64": "f64", "mixed": "fp32 z as f16 pieces (f16 main product + f16 or e5m2 correction products, "
                                              "fp32-grade) + f64 accumulate"}[main["mode"]],
            "data": "synthetic",
            "config": {"workload": cfg.name, "mode": main["mode"], "n_m": cfg.n_m, "n_b": cfg.n_b, "n_k": cfg.n_k,
                       "n_spin": cfg.n_spin, "n_o": cfg.n_o, "n_u": cfg.n_u, "n_freq": cfg.n_freq,
                       "pairs_kept": main["pairs_kept"], "credited_flop_per_step": main["flops_step"],
                       "parallelism": "replicas only" if world > 1 else "1 gpu",
                       "l2": "no flush needed: accumulator + z workspace per step far exceed the 126 MB L2"
                             if cfg.n_m >= 600 else "working set fits L2 (latency-bound config)"},
            "roofline": main["roofline"], "e2e": main["e2e"], "accuracy": main.get("accuracy"),
            **({"subset": f"first {args.n_k} of {cfg.n_k} k-points (profiling run, not a bench value)"}
               if args.n_k else {}), "gpu_launches": main["launches"],
            "clocks": main["clocks"]}
    for r in res:
        if r.get("wc"):
            line["wc"] = r["wc"]
        if r.get("sigc"):
            line["sigc"] = r["sigc"]
        if r.get("realaxis"):
            line["realaxis"] = r["realaxis"]
        if r.get("ipw"):
            line["ipw"] = r["ipw"]
        if r is not main:
            line[r["mode"]] = r
    if main.get("mixed_selection"):
        line["mixed_selection"] = main["mixed_selection"]
    if side:
        line["configs"] = side
    if world == 1 and not args.no_cpu:
        n_k_s, fsel = oracle_sample(cfg, prob, seconds_hint=args.cpu_seconds)
        dt, fl = run_oracle_sample(cfg, prob, n_k_s, fsel)
        line["cpu_baseline"] = {"value": fl / dt / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                                "sample": sample_text(cfg, n_k_s, fsel), "seconds": dt}
    print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--mode", default="both", choices=["fp64", "mixed", "both"])
    ap.add_argument("--max-n-o", type=int, default=0, help="band batch (default: whole O side)")
    ap.add_argument("--max-n-u", type=int, default=0, help="band batch (default: whole U side)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="target CPU time of the oracle sample")
    ap.add_argument("--n-k", type=int, default=0,
                    help="profiling only: run the first n_k k-points (same launch configuration); "
                         "the line is then marked config.subset and is not a bench value")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-wc", action="store_true", help="skip the W^c(i omega) leg reported beside the FP64 step")
    ap.add_argument("--no-realaxis", action="store_true", help="skip the real-axis (binned Im chi0 + Hilbert) leg")
    ap.add_argument("--no-ipw", action="store_true", help="skip the IPW block (row f4) leg")
    ap.add_argument("--no-sigc", action="store_true", help="skip the I^c (imaginary-axis self-energy) leg")
    ap.add_argument("--no-accuracy", action="store_true", help="skip the oracle check of the timed outputs")
    ap.add_argument("--no-configs", action="store_true", help="skip the side runs of the other configurations")
    return ap.parse_args(argv)


if __name__ == "__main__":
    a = parse_args()
    sys.exit(main_reference(a) if a.impl == "reference" else main_cuda(a))
