#!/usr/bin/env python
"""bench.py -- sigma-builds/s of the TDA-risp hot path on seeded synthetic systems (BASELINE.json metric).

A "step" is one pass of the whole hot path: one `risp_matvec` over a batch of m trial vectors (J + K + diagonal, all
SURVEY 8(a) rows a4-a12) with the setup (pair list, metrics, K tensors) already built and X resident in HBM.
`value` = m * K / (sum of the K device-timed steps), max over ranks; `e2e` = the same through `risp_matvec_host` (pinned HOST
buffers, H2D and D2H inside the timed region).  Between timed iterations L2 is flushed by writing a 512 MiB buffer.
The default workload is the 300-atom system (BASELINE.json configs[2], m = 30); the line also carries the metric's second
half, the wall time of the 15-root `risp_tda_solve`, the FP64 yardsticks measured in the same run (DFMA and DMMA issue rates of
the library's own micro-kernels, cuBLAS DGEMM through torch), one roofline entry per phase, and -- `also` -- a short run of the
1000-atom system (and of the 3000-atom one with --also 4,5).  N > 1: every rank owns its own batch of m vectors (the path
shards by trial vector with no collective), weak scaling.

`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload, metric and unit.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "TDA-risp sigma-builds/s (15-root wall time and % of FP64 tensor/HBM roofline alongside)"
UNIT = "sigma-builds/s"
FP64_PER_BF16 = 45.0 / 2250.0     # nominal B200 dense FP64-tensor : bf16-tensor ratio (blackwell guide: 45 TF vs 2.25 PF)
HARTREE_EV = 27.211386245988
T_START = time.time()


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained", d["bf16_tflops"]), src="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, src="fallback")


class ClockSampler:
    FIELDS = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.2] or [r for _, r in self.rows]
        if not rows:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        sm = sorted(float(r[0]) for r in rows if r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 2 + k and r[2 + k] == "Active" for r in rows)]
        return dict(sm_mhz=sm[len(sm) // 2] if sm else None, sm_max_mhz=float(rows[0][1]) if rows[0][1].replace(".", "").isdigit() else None,
                    reasons=reasons, samples=len(rows))


# ------------------------------------------------------------------------------------------------ the CPU oracle, bounded
_AUX_ATOMS_SAMPLE = {1: None, 2: None, 3: 8, 4: 1, 5: 1}      # heavy atoms whose aux shells enter the sample (None: all of them)


class OracleSample:
    """The oracle as it stands on a bounded sample of the workload: `oracle.sigma`'s three terms with the auxiliary basis
    restricted to the shells of the first few heavy atoms, timed term by term and extrapolated linearly in the number of
    auxiliary functions (J and K are sums over auxiliary functions of equally sized pieces of work, oracle.coulomb /
    oracle.exchange); configs 1-2 use the whole auxiliary basis and need no extrapolation."""

    def __init__(self, s, m_s):
        from oracle.risp_oracle import Oracle
        na = _AUX_ATOMS_SAMPLE[s["cfg"]]
        self.s, self.m_s = s, m_s
        self.full = na is None
        sub = s
        if not self.full:
            keep = np.arange(min(2 * na, len(s["aux_l"])))
            sub = dict(s)
            for k in ("aux_atom", "aux_l", "aux_exp", "aux_in_K"):
                sub[k] = np.ascontiguousarray(np.asarray(s[k])[keep])
            sub["naux"] = len(keep)
        self.o = Oracle(sub)
        t0 = time.time(); self.o.build(); self.t_build = time.time() - t0
        nJ_full = int(np.sum(2 * np.asarray(s["aux_l"]) + 1)); nK_full = int(np.sum((2 * np.asarray(s["aux_l"]) + 1) * np.asarray(s["aux_in_K"])))
        self.fJ = nJ_full / self.o.nfun(self.o.selJ)
        self.fK = nK_full / max(self.o.nfun(self.o.selK), 1)
        self.cores = os.cpu_count()

    def step(self, X):
        """one sample evaluation; returns the extrapolated seconds of a full oracle.sigma on these vectors"""
        o = self.o
        t0 = time.time(); dg = o.delta[None] * X; t_d = time.time() - t0
        t0 = time.time(); J = o.coulomb(X); t_j = time.time() - t0
        t0 = time.time(); K = o.exchange(X); t_k = time.time() - t0
        self.last = (dg, J, K)
        return t_d + self.fJ * t_j + self.fK * t_k, t_d + t_j + t_k

    def describe(self, t_cpu):
        if self.full:
            return f"oracle.sigma (all three terms) on {self.m_s} trial vectors, whole auxiliary basis, {t_cpu:.1f} s of CPU work per call; tensor build ({self.t_build:.1f} s) excluded like risp_setup"
        return (f"oracle diagonal + coulomb + exchange on {self.m_s} trial vectors with the auxiliary shells of the first {_AUX_ATOMS_SAMPLE[self.s['cfg']]} heavy "
                f"atoms ({self.o.nfun(self.o.selJ)} J / {self.o.nfun(self.o.selK)} K functions), {t_cpu:.1f} s of CPU work per call, J and K times scaled by "
                f"{self.fJ:.1f} / {self.fK:.1f} to the whole auxiliary basis; tensor build of the sample ({self.t_build:.1f} s) excluded like risp_setup")


def _fp32_mode(torch, ctx, X, sigma, flush, stream, steps, warmup, m, d, small):
    """risp_matvec with RISP_PRECISION_FP32_K: Eq. 22-23 on the tcgen05 tensor cores (three bf16 terms per operand, six MMAs per
    k step, FP32 accumulation).  Reported beside the FP64 headline, never instead of it."""
    no, nv, nK = d["noccK"], d["nvirK"], d["nauxK"]
    K64 = torch.from_numpy(ctx.stage("K", m)).to(X.device) if small else None      # K' of the FP64 step just timed
    sig64 = sigma.clone() if small else sigma.view(m, -1)[:, ::997].clone()
    ctx.set_precision(1)
    try:
        for _ in range(warmup):
            ctx.matvec(X, sigma)
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        phase = {}
        for a, b in evs:
            flush.zero_()
            a.record(stream)
            ctx.matvec(X, sigma)
            b.record(stream)
            b.synchronize()
            for k, v in ctx.timings().items():
                phase[k] = phase.get(k, 0.0) + (v if isinstance(v, float) else 0.0)
        tim = ctx.timings()
        t_dev = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
        s32 = sigma if small else sigma.view(m, -1)[:, ::997]
        out = dict(value=m * steps / t_dev, unit=UNIT, ms_per_step=1e3 * t_dev / steps, dtype="f64 integrals, J and Davidson algebra; K contractions "
                   "bf16x3 operands (24 significand bits) with FP32 accumulation on tcgen05, aux chunks summed in FP64",
                   phases_ms={k: round(1e3 * v / steps, 4) for k, v in phase.items() if k not in ("kernel_launches", "first_chunk_naux")},
                   gpu_launches=tim["kernel_launches"] * steps,
                   sigma_rel_diff_vs_fp64=float((s32 - sig64).norm() / sig64.norm()))
        if small:
            K32 = torch.from_numpy(ctx.stage("K", m)).to(X.device)
            out["K_rel_diff_vs_fp64"] = float((K32 - K64).norm() / K64.norm())
            del K32
        npf = tim["first_chunk_naux"]
        t1, t2 = phase["k_gemm1"] / steps, phase["k_gemm2"] / steps
        f1, f2 = 2.0 * m * no * nv * nv * npf, 2.0 * m * no * no * nv * npf
        # the tensor cores execute six bf16 MMAs per product: `achieved` is the executed bf16 rate, the peak is the measured bf16 one
        out["roofline"] = dict(bound="tensor", kernel="tcgemm2_bf16x3_kernel, CTA pair (Eq. 22, M^P = X' T_ab^P)", unit="TFLOP/s", achieved=6 * f1 / t1 / 1e12,
                               fp32_equivalent_tflops=f1 / t1 / 1e12, launch_ms=1e3 * t1, flops_per_launch_fp32=f1)
        out["roofline_eq23"] = dict(bound="tensor", kernel="tcgemm2_bf16x3_kernel, CTA pair (Eq. 23, K' += T_ij M)", unit="TFLOP/s", achieved=6 * f2 / t2 / 1e12,
                                    fp32_equivalent_tflops=f2 / t2 / 1e12, launch_ms=1e3 * t2, flops_per_launch_fp32=f2)
        out["k_phase_fp32_equivalent_tflops"] = 2.0 * m * nK * no * nv * (no + nv) / (phase["k_total"] / steps) / 1e12
        return out
    finally:
        ctx.set_precision(0)
        del K64, sig64


def _fp32_jk_mode(torch, ctx, X, sigma, flush, stream, steps, warmup, m, sig64):
    """risp_matvec with RISP_PRECISION_FP32_JK: the four AO<->MO transform GEMMs of the J term on the tcgen05 path as well
    (the paper keeps everything after the integrals in single precision)."""
    ctx.set_precision(2)
    try:
        for _ in range(warmup):
            ctx.matvec(X, sigma)
        torch.cuda.synchronize()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        phase = {}
        for a, b in evs:
            flush.zero_()
            a.record(stream)
            ctx.matvec(X, sigma)
            b.record(stream)
            b.synchronize()
            for k, v in ctx.timings().items():
                phase[k] = phase.get(k, 0.0) + (v if isinstance(v, float) else 0.0)
        tim = ctx.timings()
        t_dev = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
        return dict(value=m * steps / t_dev, unit=UNIT, ms_per_step=1e3 * t_dev / steps,
                    dtype="as fp32_mode, and the AO<->MO transforms of the J term (Eq. 12, 17) as bf16x3 operands on tcgen05; integrals, ERI passes, "
                          "metric solve, diagonal and Davidson algebra FP64",
                    phases_ms={k: round(1e3 * v / steps, 4) for k, v in phase.items() if k not in ("kernel_launches", "first_chunk_naux")},
                    gpu_launches=tim["kernel_launches"] * steps,
                    sigma_rel_diff_vs_fp64=float((sigma - sig64).norm() / sig64.norm()))
    finally:
        ctx.set_precision(0)


def run_reference(args):
    """The CPU oracle as the reference arm: sigma-builds/s of the oracle on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from workloads import make_system, trial_vectors
    s = make_system(args.config)
    m_s = min(args.batch if args.batch > 0 else s["m"], args.ref_vectors)
    smp = OracleSample(s, m_s)
    X = trial_vectors(s)[:m_s]
    for _ in range(args.warmup):
        smp.step(X)
    t_est = t_cpu = 0.0
    for _ in range(args.steps):
        a, b = smp.step(X)
        t_est += a; t_cpu += b
    val = m_s * args.steps / t_est
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * t_cpu / args.steps, ms_per_step_extrapolated=1e3 * t_est / args.steps,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=s["name"], m=m_s, atoms=int(s["natm"]), nao=s["nao"], nocc=s["nocc"], nvir=s["nvir"]),
                cpu_baseline=dict(value=val, unit=UNIT, cores=smp.cores, kind="oracle", sample=smp.describe(t_cpu / args.steps)),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ one configuration on the GPU
def _eri_flops_per_task():
    """FP64 thread-instructions per (shell pair, aux centre) task and pair class, counted by ncu on the pass kernels
    (profiles/eri_flops.json; flop = 2 DFMA + DMUL + DADD)."""
    p = os.path.join(ROOT, "profiles", "eri_flops.json")
    return json.load(open(p)) if os.path.exists(p) else None


def run_config(cfg, args, world, rank, local, dist, want_solve, want_cpu, steps, warmup):
    import torch
    from paper_2603_29257_b200 import setup
    from workloads import make_system, trial_vectors
    dev = torch.device(f"cuda:{local}")
    s = make_system(cfg)
    m = args.batch if (args.batch > 0 and cfg == args.config) else s["m"]
    if cfg == 5 and not (args.batch > 0 and cfg == args.config):
        m = 15          # X and sigma of 30 vectors (2 x 32 GB) do not fit beside the K tensors on a 180 GB part
    big = s["nocc"] * s["nvir"] * m > 1e9
    if big:    # 3000-atom scale: one pinned copy of X on the host, filled in place
        Xp = torch.empty((m, s["nocc"], s["nvir"]), dtype=torch.float64, pin_memory=True)
        X_h = trial_vectors(s, m, base_seed=260329257 + 17 * rank, out=Xp.numpy())
    else:
        X_h = trial_vectors(s, m, base_seed=260329257 + 17 * rank)
        Xp = None
    t0 = time.time()
    ctx = setup(s, device=local, max_batch=m, host_budget_bytes=args.host_budget_gb << 30)
    t_setup = time.time() - t0
    X = torch.from_numpy(X_h).to(dev)
    sigma = torch.empty_like(X)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing
    for _ in range(warmup):
        ctx.matvec(X, sigma)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    tw0 = time.time()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    phase = {}
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        ctx.matvec(X, sigma)
        b.record(stream)
        b.synchronize()
        for k, v in ctx.timings().items():
            phase[k] = phase.get(k, 0.0) + (v if isinstance(v, float) else 0.0)
    barrier()
    tw1 = time.time()
    clocks = sampler.stop(tw0, tw1) if sampler else None
    t_dev = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    tim = ctx.timings()
    d = ctx.dims()
    launches = tim["kernel_launches"] * steps

    # ---- the single-precision mode of the K contractions, same batch, same timing rules
    fp32 = fp32_jk = None
    if rank == 0 and world == 1 and not args.no_fp32 and d["nauxK"] > 0 and (cfg <= 3 or args.fp32_large):
        sig64_keep = sigma.clone() if cfg <= 4 else None
        fp32 = _fp32_mode(torch, ctx, X, sigma, flush, stream, steps, warmup, m, d, small=cfg <= 3)
        if cfg <= 4:
            fp32_jk = _fp32_jk_mode(torch, ctx, X, sigma, flush, stream, steps, warmup, m, sig64_keep)
            fp32_jk["j_sub_batch"] = ctx.dims()["j_sub_batch"]
        del sig64_keep

    # ---- end to end: pinned host buffers through risp_matvec_host
    fp = None
    sig_h = None if big else sigma.cpu().numpy()
    if big:    # the library's own staging copies of X and sigma take the place of the caller's device tensors
        fp = sigma.view(m, -1)[:, ::997].cpu()
        del X, sigma
        torch.cuda.empty_cache()
    if Xp is None:
        Xp = torch.from_numpy(X_h).pin_memory()
    Sp = torch.empty(Xp.shape, dtype=torch.float64, pin_memory=True)
    for _ in range(0 if args.no_e2e else (2 if cfg <= 3 else 1)):
        ctx.matvec_host_ptr(m, Xp.data_ptr(), Sp.data_ptr())
    barrier()
    t_e2e = 0.0
    e2e_steps = steps if cfg <= 3 else 1
    for _ in range(0 if args.no_e2e else e2e_steps):
        flush.zero_(); torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        ctx.matvec_host_ptr(m, Xp.data_ptr(), Sp.data_ptr())
        t_e2e += time.perf_counter() - t0
    barrier()
    if world > 1:
        tt = torch.tensor([t_dev, t_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_dev, t_e2e = float(tt[0]), float(tt[1])
    same = None if args.no_e2e else (bool(torch.equal(Sp.view(m, -1)[:, ::997], fp)) if big else bool(np.array_equal(Sp.numpy(), sig_h)))
    if not big:
        del X, sigma
    del flush, Xp, Sp, fp
    torch.cuda.empty_cache()

    res = None
    if rank == 0:
        pk = _peaks()
        no, nv, nK = d["noccK"], d["nvirK"], d["nauxK"]
        ms_step = 1e3 * t_dev / steps
        # a launch inside a step of a second or more runs under the sustained power / clock state, a short step under the burst one
        long_step = ms_step >= 1000.0
        bf16 = pk["bf16_sustained"] if long_step else pk["bf16"]
        peak = bf16 * FP64_PER_BF16
        peak_src = f"{pk['src']} bf16 {'sustained' if long_step else 'burst'} {bf16} TFLOP/s x nominal FP64:bf16 ratio 45/2250 ({'step >= 1 s' if long_step else 'step < 1 s'})"
        # dominant kernel: the DMMA GEMM launch M^P = X' T_ab^P (Eq. 22) of the first aux chunk
        npf = tim["first_chunk_naux"]
        flops_launch = 2.0 * m * no * nv * nv * npf
        t_launch = phase["k_gemm1"] / steps
        achieved = flops_launch / t_launch / 1e12 if t_launch > 0 else 0.0
        traffic = None
        tpath = os.path.join(ROOT, "profiles", f"traffic_cfg{cfg}.json")
        if os.path.exists(tpath):
            traffic = json.load(open(tpath)).get("dgemm_k_gemm1_dram_bytes_per_launch")
        # yardsticks measured now, on this GPU, by the library's own register-resident micro-kernels and by cuBLAS through torch
        dfma = ctx.yardstick(0, reps=3) / 1e12
        dmma = ctx.yardstick(1, reps=3) / 1e12
        A = torch.randn((8192, 8192), dtype=torch.float64, device=dev)
        for _ in range(2):
            A @ A
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); C3 = [A @ A for _ in range(3)]; e1.record(); e1.synchronize()
        cublas = 3 * 2.0 * 8192 ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12
        del A, C3
        torch.cuda.empty_cache()
        z_pairs = d["n_ao_pairs_kept"]
        flops_step = dict(K=2.0 * m * nK * no * nv * (no + nv),
                          transforms_dense=4.0 * m * s["nocc"] * s["nvir"] * s["nao"] + 4.0 * m * s["nao"] ** 2 * s["nocc"],
                          transforms_pair_sparse=4.0 * m * s["nocc"] * s["nvir"] * s["nao"] + 8.0 * m * z_pairs * s["nocc"])
        eri = _eri_flops_per_task()
        eri_entry = dict(phase="ERI passes (Eq. 14, 16): FP64 flops executed, both passes (integral generation: 2 DFMA + DMUL + DADD per task from ncu; contraction: DMMA, 2 m flops per integral)", bound="alu", unit="TFLOP/s", achieved=None, peak=dfma,
                         peak_source="risp_debug_yardstick(0): register-resident DFMA chains on all SMs, measured in this run")
        t_eri = (phase["j_pass1"] + phase["j_pass2"]) / steps
        if eri is not None and t_eri > 0:
            fl = 0.0
            ne_class = [1, 4, 9, 6, 16, 31]           # e0 components of the classes ss, ps, pp, ds, dp, dd
            mcols = 8 * ((m + 7) // 8)                # trial-vector columns the DMMA contraction really computes
            for c, npairs in enumerate(d["pairs_per_class"]):
                for ps in ("pass1", "pass2"):
                    fl += (eri[ps][c] + 2.0 * mcols * 4 * ne_class[c]) * npairs * d["n_aux_centres"]
            eri_entry.update(achieved=fl / t_eri / 1e12, frac=fl / t_eri / 1e12 / dfma, flops_per_step=fl,
                             note=eri.get("note", ""))
        t_tr = (phase["j_transform_in"] + phase["j_transform_out"]) / steps
        line = dict(
            metric=METRIC, value=world * m * steps / t_dev, unit=UNIT, n_gpus=world, steps=steps, warmup=warmup,
            ms_per_step=ms_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
            config=dict(workload=s["name"], m=m, atoms=int(s["natm"]), nao=s["nao"], nocc=s["nocc"], nvir=s["nvir"], nauxJ=d["nauxJ"], nauxK=nK,
                        noccK=no, nvirK=nv, shell_pairs_kept=d["n_shell_pairs_kept"], shell_pairs=d["n_shell_pairs"], pairs_per_class=list(d["pairs_per_class"]), aux_centres=d["n_aux_centres"],
                        ao_pair_survival=round(2.0 * d["n_ao_pairs_kept"] / (s["nao"] * (s["nao"] + 1)), 4),
                        K_tensors=f"packed lower triangles; {d['nauxK_device']} of {nK} aux slices in HBM, {d['bytes_T_host']} B in pinned host memory",
                        bytes_T=d["bytes_Tij"] + d["bytes_Tab"], aux_chunk=d["aux_chunk"], j_sub_batch=d["j_sub_batch"], j_panels=d["j_panels"],
                        l2="flushed between steps (512 MiB write)",
                        parallelism=f"trial-vector shards x{world}", setup_s=round(t_setup, 3)),
            clocks=clocks,
            e2e=None if args.no_e2e else dict(value=world * m * e2e_steps / t_e2e, steps=e2e_steps, unit=UNIT, h2d_bytes_per_step=int(X_h.nbytes), d2h_bytes_per_step=int(X_h.nbytes),
                     bitwise_equal_to_device_path=same),
            gpu_launches=launches,
            roofline=dict(bound="tensor", kernel="dgemm_tma_kernel<KC,KC,MI> (K contraction M^P = X' T_ab^P, Eq. 22)", achieved=achieved, peak=peak,
                          unit="TFLOP/s", frac=achieved / peak, traffic=traffic, peak_source=peak_src,
                          context=dict(dmma_issue_ceiling_tflops_measured=dmma, cublas_dgemm_8192_tflops_measured=cublas, dfma_tflops_measured=dfma,
                                       frac_of_dmma_ceiling=achieved / dmma, frac_of_cublas_dgemm=achieved / cublas,
                                       note="FP64 tensor op of sm_100a is the warp-level DMMA.8x8x4; `peak` follows the tier rule (another dtype's "
                                            "measured peak x nominal ratio), the three yardsticks beside it were measured in this run"),
                          flops_per_launch=flops_launch, launch_ms=1e3 * t_launch),
            phases_ms={k: round(1e3 * v / steps, 4) for k, v in phase.items() if k not in ("kernel_launches", "first_chunk_naux")},
            rooflines_other=[
                dict(phase="K contraction, all chunks (Eq. 22-23, packed-slice expansion included)", bound="tensor", unit="TFLOP/s",
                     achieved=flops_step["K"] / (phase["k_total"] / steps) / 1e12 if phase.get("k_total") else None, peak=peak,
                     frac=flops_step["K"] / (phase["k_total"] / steps) / 1e12 / peak if phase.get("k_total") else None),
                dict(phase="J AO<->MO transforms (Eq. 12, 17; e0 gather/scatter and the diagonal term included), against the PAIR-SPARSE flop count "
                           "4 m nocc nvir nao + 8 m z nocc the method needs", bound="tensor", unit="TFLOP/s",
                     achieved=flops_step["transforms_pair_sparse"] / t_tr / 1e12, peak=peak, frac=flops_step["transforms_pair_sparse"] / t_tr / 1e12 / peak,
                     executed_tflops=flops_step["transforms_dense"] / t_tr / 1e12),
                dict(phase="sigma[window] -= K' (Eq. 10)", bound="hbm", unit="GB/s",
                     achieved=24.0 * m * no * nv / (phase["assemble"] / steps) / 1e9 if phase.get("assemble") else None, peak=pk["hbm"],
                     frac=24.0 * m * no * nv / (phase["assemble"] / steps) / 1e9 / pk["hbm"] if phase.get("assemble") else None),
                eri_entry,
            ],
            flops_per_step=flops_step,
        )
        if fp32 is not None:
            pk16 = pk["bf16_sustained"] if fp32["ms_per_step"] >= 1000.0 else pk["bf16"]
            for key in ("roofline", "roofline_eq23"):
                r = fp32[key]
                r["peak"] = pk16; r["frac"] = r["achieved"] / pk16
                r["peak_source"] = f"{pk['src']} bf16 cuBLAS throughput ({'sustained' if fp32['ms_per_step'] >= 1000.0 else 'burst'})"
            line["fp32_mode"] = fp32
            if fp32_jk is not None:
                line["fp32_jk_mode"] = fp32_jk
        smp = None
        if want_cpu and world == 1 and cfg <= 4:
            ms_ = min(m, 30 if cfg <= 2 else args.ref_vectors)
            smp = OracleSample(s, ms_)
            t_est, t_cpu = smp.step(X_h[:ms_])
            cb = dict(value=ms_ / t_est, unit=UNIT, cores=smp.cores, kind="oracle", sample=smp.describe(t_cpu))
            if smp.full:
                ref = smp.last[0] + 2.0 * smp.last[1] - smp.last[2]
                cb["gpu_vs_oracle_rel_err"] = float(np.linalg.norm(sig_h[:ms_] - ref) / np.linalg.norm(ref))
            line["cpu_baseline"] = cb
        if want_solve:
            big_dim = s["nocc"] * s["nvir"] >= 5e7
            kw = dict(tol=args.solve_tol, max_iter=args.solve_max_iter, allow_unconverged=True, n_guess=args.solve_n_guess, max_seconds=args.solve_max_seconds)
            flags = (8 if args.solve_fp32_host else 0) | (16 if big_dim else 0) | (32 if args.progress_file else 0)
            if args.solve_mode == "fp32":      # the whole solve (and the residual re-check) in the single-precision mode of the K contractions
                ctx.set_precision(1)
            omega, Xs, info = ctx.tda_solve(s["nroots"], want_vectors=True, flags=flags, **kw)
            sv = dict(precision="fp32_k" if args.solve_mode == "fp32" else "fp64", nroots=s["nroots"], tol=args.solve_tol, n_guess=args.solve_n_guess or 2 * s["nroots"], wall_s=info["sec_total"], matvec_s=info["sec_matvec"],
                      alloc_s=info["sec_alloc"], subspace_s=info["sec_subspace"], block=info["block"], capacity=info["capacity"],
                      cached_vectors=info["cached_vectors"], host_subspace_gb=info["bytes_host_subspace"] / 1e9,
                      host_store="fp32" if args.solve_fp32_host else "fp64", iterations=info["iterations"], n_sigma=info["n_sigma"],
                      restarts=info["restarts"], converged=info["converged"], subspace_max=info["subspace_max"], resid_max=float(max(info["resid"])),
                      omega_ev=[float(x) * HARTREE_EV for x in omega], h2d_gb=info["bytes_h2d"] / 1e9, d2h_gb=info["bytes_d2h"] / 1e9,
                      setup_s=round(t_setup, 3), setup_plus_solve_s=round(t_setup + info["sec_total"], 3))
            if args.progress_file:      # a long solve leaves its record behind even if something after it fails
                json.dump(sv, open(args.progress_file, "w"))
            # compositional check (v) of SURVEY 8(c).6: residuals ||A x_k - omega_k x_k|| recomputed by fresh risp_matvec calls
            try:
                rmax, blk = 0.0, info["block"]
                for c0 in range(0, s["nroots"], blk):
                    Xc = (torch.from_numpy(Xs[c0:c0 + blk]).to(dev) if big_dim else Xs[c0:c0 + blk].contiguous())
                    AX = ctx.matvec(Xc)
                    r = (AX - torch.from_numpy(omega[c0:c0 + blk]).to(dev)[:, None, None] * Xc).reshape(Xc.shape[0], -1).norm(dim=1)
                    rmax = max(rmax, float(r.max()))
                    del AX, Xc
                sv["resid_recomputed_max"] = rmax
            except Exception as e:      # reported, not hidden
                sv["resid_recomputed_error"] = repr(e)
            del Xs
            ctx.set_precision(0)
            if smp is not None and smp.full and cfg <= 2:      # the CPU oracle's own Davidson on the same problem (same tolerance)
                t0 = time.time()
                th_ref, _, iref = smp.o.davidson(s["nroots"], tol=args.solve_tol)
                sv["cpu_oracle"] = dict(wall_s=time.time() - t0, iterations=int(iref["iterations"]), n_sigma=int(iref["n_sigma"]),
                                        converged=bool(iref["converged"]), cores=os.cpu_count(),
                                        max_abs_diff_ev=float(np.abs(np.asarray(omega) - th_ref).max() * HARTREE_EV))
            elif "cpu_baseline" in line:
                sv["cpu_oracle_estimate"] = dict(wall_s=info["n_sigma"] / line["cpu_baseline"]["value"], cores=os.cpu_count(),
                                                 note="n_sigma of the GPU solve / sampled oracle sigma-builds/s; the oracle's own Davidson is not run at this size")
            line["solve"] = sv
            if fp32 is not None and not big_dim and args.solve_mode == "both" and cfg <= 3:
                ctx.set_precision(1)
                try:
                    om32, _, i32 = ctx.tda_solve(s["nroots"], want_vectors=False, flags=flags & ~32, **kw)
                    fp32["solve"] = dict(wall_s=i32["sec_total"], matvec_s=i32["sec_matvec"], iterations=i32["iterations"], n_sigma=i32["n_sigma"],
                                         converged=i32["converged"], resid_max=float(max(i32["resid"])), tol=args.solve_tol,
                                         max_abs_diff_vs_fp64_solve_ev=float(np.abs(np.asarray(om32) - np.asarray(omega)).max() * HARTREE_EV))
                finally:
                    ctx.set_precision(0)
                if fp32_jk is not None:
                    ctx.set_precision(2)
                    try:
                        omjk, _, ijk = ctx.tda_solve(s["nroots"], want_vectors=False, flags=flags & ~32, **kw)
                        fp32_jk["solve"] = dict(wall_s=ijk["sec_total"], matvec_s=ijk["sec_matvec"], iterations=ijk["iterations"], n_sigma=ijk["n_sigma"],
                                                converged=ijk["converged"], resid_max=float(max(ijk["resid"])), tol=args.solve_tol,
                                                max_abs_diff_vs_fp64_solve_ev=float(np.abs(np.asarray(omjk) - np.asarray(omega)).max() * HARTREE_EV))
                    finally:
                        ctx.set_precision(0)
        res = line
    ctx.close()
    del ctx
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    return res


def run_sharded(args, world, rank, local, dist):
    """--parallel shard (N > 1): ONE problem, P-sharded over the ranks: every rank holds 1/N of the shell pairs
    and of the K-tensor slices, X is replicated, two all-reduces per batch (R between the integral passes, sigma at the end).
    Strong scaling: the same m sigma-builds are done by all ranks together."""
    import torch
    from paper_2603_29257_b200 import setup
    from paper_2603_29257_b200.sharded import sharded_matvec
    from workloads import make_system, trial_vectors
    dev = torch.device(f"cuda:{local}")
    s = make_system(args.config)
    m = min(args.batch if args.batch > 0 else s["m"], 32)
    X = torch.from_numpy(trial_vectors(s, m)).to(dev)
    t0 = time.time()
    ctx = setup(s, device=local, max_batch=m, shard_rank=rank, shard_count=world)
    t_setup = time.time() - t0
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)
    for _ in range(args.warmup):
        sharded_matvec(ctx, X)
    dist.barrier(); torch.cuda.synchronize(dev)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in evs:
        flush.zero_()
        dist.barrier()
        a.record(stream)
        sig = sharded_matvec(ctx, X)
        b.record(stream)
        b.synchronize()
    dist.barrier(); torch.cuda.synchronize(dev)
    tt = torch.tensor([sum(a.elapsed_time(b) for a, b in evs) * 1e-3], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    d = ctx.dims()
    launches = ctx.timings()["kernel_launches"] * args.steps
    ctx.close()
    if rank == 0:
        t_dev = float(tt[0])
        print(json.dumps(dict(metric=METRIC, value=m * args.steps / t_dev, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                              ms_per_step=1e3 * t_dev / args.steps, higher_is_better=True, scaling="strong", vs_baseline=None, dtype="f64", data="synthetic",
                              config=dict(workload=s["name"], m=m, atoms=int(s["natm"]), nao=s["nao"], nocc=s["nocc"], nvir=s["nvir"],
                                          parallelism=f"P-sharded x{world}: shell pairs and K aux centres dealt round robin, all-reduce of R and of sigma",
                                          shell_pairs_kept_rank0=d["n_shell_pairs_kept"], nauxK_rank0=d["nauxK"], setup_s=round(t_setup, 3),
                                          l2="flushed between steps (512 MiB write)"),
                              gpu_launches=launches, e2e=None, roofline=None, cpu_baseline=None,
                              note="sharded mode: device-resident replicated X; no roofline / e2e legs in this mode")))


def run_extras(args):
    """--extras: the follow-on rows of the path on the chosen workload, one JSON line of its own: the full-TDDFT
    product ((A+B) X, (A-B) X) per second, the 15-root risp_tddft_solve, and risp_transition_properties of the TDA roots.  Reported
    beside the headline, not part of it."""
    import torch
    from paper_2603_29257_b200 import setup
    from workloads import make_system, trial_vectors
    s = make_system(args.config)
    m = args.batch if args.batch > 0 else s["m"]
    dev = torch.device("cuda:0")
    t0 = time.time()
    ctx = setup(s, flags=8, max_batch=m)                      # RISP_FLAG_TDDFT: also builds T_ia^P over the window
    t_setup = time.time() - t0
    X = torch.from_numpy(trial_vectors(s, m)).to(dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)
    for _ in range(max(args.warmup, 3)):
        ctx.matvec_tddft(X)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in evs:
        flush.zero_()
        a.record(stream)
        sp, sm = ctx.matvec_tddft(X)
        b.record(stream)
        b.synchronize()
    t_td = sum(a.elapsed_time(b) for a, b in evs) * 1e-3
    launches = ctx.timings()["kernel_launches"]
    sig = ctx.matvec(X)
    # A = ((A+B) + (A-B)) / 2: the TDA product of the same context must be the mean of the two TDDFT products
    mean_err = float(((0.5 * (sp + sm)) - sig).norm() / sig.norm())
    del sp, sm, sig
    n = s["nroots"]
    om, Xr, info = ctx.tda_solve(n, tol=args.solve_tol, max_iter=args.solve_max_iter, want_vectors=True, allow_unconverged=True)
    ctx.transition_properties(Xr, om)
    t0 = time.perf_counter()
    for _ in range(3):
        mu, mm, f, R = ctx.transition_properties(Xr, om)
    t_prop = (time.perf_counter() - t0) / 3
    del Xr
    Om, _, _, tinfo = ctx.tddft_solve(n, tol=args.solve_tol, max_iter=args.solve_max_iter, allow_unconverged=True)
    d = ctx.dims()
    ctx.close()
    no, nv, nK = d["noccK"], d["nvirK"], d["nauxK"]
    print(json.dumps(dict(
        impl="extras", workload=s["name"], m=m, dtype="f64", data="synthetic", setup_s=round(t_setup, 3),
        tddft_matvec=dict(value=m * args.steps / t_td, unit="(A+B, A-B) product pairs/s", ms_per_step=1e3 * t_td / args.steps, steps=args.steps,
                          gpu_launches_per_step=launches, extra_flops_vs_tda=4.0 * m * nK * no * no * nv,
                          tda_product_is_mean_of_both_rel_err=mean_err, l2="flushed between steps (512 MiB write)"),
        tda_solve=dict(wall_s=info["sec_total"], iterations=info["iterations"], n_sigma=info["n_sigma"], converged=info["converged"]),
        tddft_solve=dict(nroots=n, tol=args.solve_tol, wall_s=tinfo["sec_total"], matvec_s=tinfo["sec_matvec"], iterations=tinfo["iterations"],
                         n_sigma=tinfo["n_sigma"], converged=tinfo["converged"], resid_max=float(max(tinfo["resid"])),
                         omega_ev=[float(x) * HARTREE_EV for x in Om],
                         max_tda_minus_tddft_ev=float(np.max(om - Om) * HARTREE_EV), min_tda_minus_tddft_ev=float(np.min(om - Om) * HARTREE_EV)),
        transition_properties=dict(states=n, ms_per_call=1e3 * t_prop, oscillator_strengths=[float(x) for x in f],
                                   rotatory_strengths=[float(x) for x in R]))))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="risp", choices=["risp", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index + 1 (default 3: the 300-atom system)")
    ap.add_argument("--ref-vectors", type=int, default=10, help="trial vectors per step of the CPU oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--batch", type=int, default=0, help="trial vectors per step (0: the config's m)")
    ap.add_argument("--solve-max-iter", type=int, default=150)
    ap.add_argument("--solve-tol", type=float, default=1e-5)
    ap.add_argument("--solve-max-seconds", type=int, default=0, help="wall-clock guard of the solve (0: none)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (long runs under a wall-clock limit)")
    ap.add_argument("--solve-n-guess", type=int, default=0, help="initial unit vectors of the solve (0: 2 * nroots, the config's batch of 30)")
    ap.add_argument("--solve-fp32-host", action="store_true", help="RISP_SOLVE_HOST_FP32 for the solve of the 1000/3000-atom systems")
    ap.add_argument("--progress-file", default="", help="write the solve record to this file as soon as risp_tda_solve returns")
    ap.add_argument("--no-solve", action="store_true", help="skip the 15-root risp_tda_solve")
    ap.add_argument("--solve-mode", default="both", choices=["both", "fp64", "fp32"],
                    help="both: FP64 solve, then (300 atoms and below) the same solve in the single-precision mode; fp32: only the latter")
    ap.add_argument("--no-fp32", action="store_true", help="skip the single-precision-mode leg (RISP_PRECISION_FP32_K)")
    ap.add_argument("--fp32-large", action="store_true", help="run the single-precision-mode leg on the 1000/3000-atom systems too")
    ap.add_argument("--solve", action="store_true", help="(default) kept for compatibility")
    ap.add_argument("--also", default="4", help="comma separated further configs run briefly after the main one (1 GPU only); '' for none")
    ap.add_argument("--also-budget-s", type=float, default=420.0, help="an `also` config starts only if the run is younger than this")
    ap.add_argument("--parallel", default="vectors", choices=["vectors", "shard"],
                    help="N > 1: 'vectors' = every rank its own batch (weak scaling, no collective); 'shard' = one P-sharded problem (strong scaling)")
    ap.add_argument("--extras", action="store_true", help="instead of the headline: full-TDDFT products and solve, transition properties (one JSON line)")
    ap.add_argument("--host-budget-gb", type=int, default=0, help="pinned-host budget of the Davidson subspace (0: half of the host memory)")
    args = ap.parse_args()
    # contract: >= 3 warm-up steps; the 1000/3000-atom configs (tens of seconds to minutes per step) are allowed 1 and say so
    args.warmup = (max(args.warmup, 3) if args.config <= 3 else max(args.warmup, 1)) if args.impl == "risp" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if args.extras:
        if rank == 0:
            run_extras(args)
        return
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    if world > 1 and args.parallel == "shard":
        run_sharded(args, world, rank, local, dist)
        dist.destroy_process_group()
        return
    solve_main = not args.no_solve and world == 1 and args.config <= 4
    solve_main = solve_main or (not args.no_solve and world == 1 and args.solve)
    line = run_config(args.config, args, world, rank, local, dist, want_solve=solve_main, want_cpu=not args.no_cpu_baseline,
                      steps=args.steps, warmup=args.warmup)
    if rank == 0 and world == 1 and args.also:
        line["also"] = []
        for c in [int(x) for x in args.also.split(",") if x.strip()]:
            if c == args.config:
                continue
            if time.time() - T_START > args.also_budget_s:
                line["also"].append(dict(workload=f"cfg{c}", skipped=f"run already {time.time() - T_START:.0f} s old (budget {args.also_budget_s:.0f} s)"))
                continue
            sub = run_config(c, args, 1, 0, local, dist, want_solve=False, want_cpu=False, steps=2 if c == 4 else 1, warmup=1)
            keep = {k: sub[k] for k in ("value", "unit", "steps", "warmup", "ms_per_step", "config", "e2e", "roofline", "phases_ms", "rooflines_other", "clocks")}
            line["also"].append(keep)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
