#!/usr/bin/env python
"""bench.py -- throughput of the odd-even Wilson-clover hot path on B200 (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5]

Workload (BASELINE.json north_star / configs[4]): 64^3 x 128 lattice, fp32, links
exp(i*0.5*H) re-unitarised, csw = 1.5, m0 = -0.2, antiperiodic time; one STEP = one call of
the fused Richardson smoother  ddamg_richardson(nu = 4, omega = 0.9)  on a Gaussian rhs and a
non-zero Gaussian initial guess (so that every sweep is a full Schur apply): rows a2-a7 of
the hot path.  The remaining rows are timed beside it in the same run and reported under
"rows": the plain Schur apply (GB/s, GFLOP/s: BASELINE.json's metric), the whole eq.-2
smoother call (a10: prepare_rhs + sweeps + reconstruct_odd), GMRES(1,10) (a8, a9) and the
setup steps (a0, a1).

value      = V * nu * N / t   [site-sweeps/s], inputs resident in HBM, CUDA events per step
e2e        = same metric through the public API with HOST (pinned) buffers: H2D of b_e and
             x^(0), the call, D2H of x^(nu) inside the timed region
roofline   = dominant kernel (B': A_ee x - H_eo t + Richardson update), algorithmic bytes
             1248 B/even site / CUDA-event duration, against MEASURED_PEAKS.json
cpu_baseline = the fp64 oracle (oracle/, as it stands) timed on the host cores on a bounded
             sample (16^3 x 32 lattice, same recipe)
Multi-GPU: the path does not shard in this build ("replicas only"): --gpus N runs
N independent replicas, one per rank, no data-path collective; scaling = "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CONFIGS = {
    # cfg: L, T, eps, reunit, csw, m0, bc, omega
    2: dict(L=16, T=16, eps=0.3, reunit=False, csw=1.0, m0=-0.1, bc=1, omega=1.0),
    3: dict(L=32, T=64, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
    4: dict(L=48, T=96, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
    5: dict(L=64, T=128, eps=0.5, reunit=True, csw=1.5, m0=-0.2, bc=1, omega=0.9),
}
NU = 4
# algorithmic bytes per EVEN site, fp32, 18-real links
BYTES_A = 1056          # kernel A : 8 links 576 + x_e neighbours 96 + A_oo^-1 288 + write 96
BYTES_B = 1152          # kernel B : 8 links 576 + t_o 96 + x_e 96 + A_ee 288 + write 96
BYTES_BR = 1248         # kernel B': kernel B + b_e 96
FLOP_PER_SITE = 1824    # 1320 (hop) + 504 (2 x 6x6 Hermitian mat-vec), per lattice site
# dram__bytes_read.sum + dram__bytes_write.sum per launch of kernel B' at config 5, from the
# ncu --set full capture summarised in profiles/ (None until a capture exists)
NCU_TRAFFIC_BYTES = {18: {5: 21.274e9}, 12: {5: 18.073e9}}     # profiles/r1b_ncu_full_dslash.md, profiles/r1d_ncu_full_dslash12.md
CPU_SAMPLE = dict(L=16, T=32)
# SAP(n, m) row: the paper's smoother parameters (Tables 1, 2, 6) on 4^4 blocks
SAP_N, SAP_M, SAP_BLOCK = 3, 4, (4, 4, 4, 4)
SAP_HOP_FLOP = 990      # in-block hopping sum: on a 4^4 block 6 of the 8 neighbours are inside on average (1320 * 6/8)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def wait_ready(self, timeout_s: float = 5.0):
        """Block until nvidia-smi has delivered its first sample (its start-up takes longer than a short
        timed region), then forget the idle samples: everything kept is from the warm-up on."""
        t0 = time.perf_counter()
        while self.proc and not self.rows and time.perf_counter() - t0 < timeout_s:
            time.sleep(0.02)
        self.rows.clear()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except Exception:
                continue
            for name, col in (("hw_slowdown", 5), ("hw_thermal_slowdown", 6), ("sw_thermal_slowdown", 7),
                              ("sw_power_cap", 8)):
                if len(r) > col and r[col].lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- multi-rank host logic
def max_over_ranks(ms: float, world: int, device="cpu") -> float:
    """Timed-region length of the whole job = MAX over ranks (replicas run concurrently)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(V: int, nu: int, world: int, ms_per_step: float) -> float:
    """Whole-job site-sweeps/s: every rank sweeps its own replica of the V-site lattice nu times."""
    return V * nu * world / (ms_per_step * 1e-3)


# --------------------------------------------------------------------------- reference arm
def oracle_run(steps: int, warmup: int, cfg: int):
    """The CPU oracle as it stands, Richardson nu=4 on a bounded sample of the workload."""
    import numpy as np
    import gen
    import oracle
    c = CONFIGS[cfg]
    L, T = CPU_SAMPLE["L"], CPU_SAMPLE["T"]
    U = gen.gauge_field(L, T, 1000 + cfg, c["eps"], c["reunit"]).numpy()
    op = oracle.WilsonClover(L, T, c["csw"], c["m0"], c["bc"], U)
    b = np.where(op.even, gen.spinor_field(L, T, 2000 + cfg).numpy(), 0.0)
    x0 = np.where(op.even, gen.spinor_field(L, T, 2500 + cfg).numpy(), 0.0)
    for _ in range(warmup):
        oracle.richardson(op.apply_schur, b, x0, NU, c["omega"])
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.richardson(op.apply_schur, b, x0, NU, c["omega"])
    dt = time.perf_counter() - t0
    V = L * L * L * T
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return dict(value=V * NU * steps / dt, ms_per_step=1e3 * dt / steps, cores=cores,
                sample=f"{L}^3x{T} lattice (config {cfg} recipe), {steps} calls of Richardson nu={NU}, fp64 oracle, OpenMP over sites")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    c = CONFIGS[cfg]
    steps = max(1, min(args.steps, 40))
    r = oracle_run(steps, max(1, min(args.warmup, 3)), cfg)
    line = {
        "impl": "reference", "metric": "Richardson sites/s (odd-even Schur Wilson-clover, nu=4)",
        "value": r["value"], "unit": "site-sweeps/s", "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup,
        "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {cfg}: {c['L']}^3x{c['T']} Wilson-clover csw={c['csw']} m0={c['m0']}, "
                               f"Richardson nu={NU} omega={c['omega']}; bounded CPU sample {r['sample']}"},
        "cpu_baseline": {"value": r["value"], "unit": "site-sweeps/s", "cores": r["cores"], "kind": "oracle",
                         "sample": r["sample"]},
        "e2e": {"value": r["value"], "unit": "site-sweeps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------- our arm
def f64_apply_row(torch, gen, Ddamg, dev):
    """fp64 Schur apply at 48^3 x 96 (config 4 recipe, 18-real links): the precision of BASELINE.json's
    fp64 parity bar, timed against the two-pass byte model at 8 bytes per real (4416 B per even site)."""
    from paper_2407_08092_b200 import F64
    c = CONFIGS[4]
    L, T = c["L"], c["T"]
    ctx = Ddamg(L, T, c["csw"], c["m0"], c["bc"], F64, stream=None, device=dev)
    U = gen.gauge_field(L, T, 1004, c["eps"], c["reunit"], device=dev, dtype=torch.complex128)
    ctx.load_gauge(U)
    ctx.build_clover()
    del U
    x, _ = ctx.pack(gen.spinor_field(L, T, 2004, device=dev, dtype=torch.complex128))
    y = ctx.half_spinor()
    for _ in range(3):
        ctx.apply_schur(x, y)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n = 10
    a.record()
    for _ in range(n):
        ctx.apply_schur(x, y)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b) / n
    V = L * L * L * T
    peak, _ = _peaks()
    gbs = 2 * 2208 * (V // 2) / (ms * 1e-3) / 1e9
    ctx.close()
    return {"lattice": "48^3x96, fp64, 18-real links", "ms": ms, "sites_per_s": V / (ms * 1e-3),
            "GBps_two_pass_model": gbs, "frac_of_peak": gbs / peak,
            "GFLOPps": (FLOP_PER_SITE * V + 24 * (V // 2)) / (ms * 1e-3) / 1e9}


def paper_context_row(torch, gen, Ddamg, F32, dev, recon):
    """One smoother call each of odd-even Richardson(12, 1.5), odd-even GMRES(3, 4) and SAP(3, 4) at 48^3 x 96."""
    c = CONFIGS[4]
    L, T = c["L"], c["T"]
    ctx = Ddamg(L, T, c["csw"], c["m0"], c["bc"], F32, stream=None, device=dev)
    U = gen.gauge_field(L, T, 1004, c["eps"], c["reunit"], device=dev, dtype=torch.complex64)
    ctx.load_gauge(U)
    ctx.build_clover()
    del U
    if recon == 12:
        ctx.set_option("gauge_recon", 12)
    b_e, b_o = ctx.pack(gen.spinor_field(L, T, 2004, device=dev, dtype=torch.complex64))
    v = b_e.clone()
    lam = ctx.power_iteration(v, 10)              # Alg. 4 line 1: omega = delta / |lambda_max|, delta = 1.5
    omega = 1.5 / lam
    bhat, x_e, x_o = ctx.half_spinor(), ctx.half_spinor(), ctx.half_spinor()

    def timed_call(fn, n=5):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n

    def rich():
        ctx.prepare_rhs(b_e, b_o, bhat)
        ctx.richardson(bhat, x_e, 12, omega, zero_init=True)
        ctx.reconstruct_odd(b_o, x_e, x_o)

    def gm():
        ctx.prepare_rhs(b_e, b_o, bhat)
        ctx.gmres_oe(bhat, x_e, 4, 3, zero_init=True)
        ctx.reconstruct_odd(b_o, x_e, x_o)

    def sap():
        ctx.sap(b_e, b_o, x_e, x_o, 3, 4, block=(4, 4, 4, 4), zero_init=True)

    out = {"lattice": "48^3x96 (the paper's 96x48^3 shape), synthetic links, fp32, one B200",
           "omega_power_iteration": omega,
           "odd_even_richardson_12_ms": timed_call(rich), "odd_even_gmres_3x4_ms": timed_call(gm),
           "sap_3x4_ms": timed_call(sap),
           "paper_gpu_ms": {"odd_even_richardson": 360.0, "odd_even_gmres_3x4": 450.0, "sap_3x4": 330.0},
           "paper_cpu_ms": {"odd_even_richardson": 4800.0, "odd_even_gmres_3x4": 5660.0, "sap_3x4": 4390.0},
           "paper_hardware": "Table 2, PAPER.md:258-262: 4 ORISE nodes, 16 GPUs (64 SMs, 16 GB HBM2, HIP, host-staged halos) "
                             "/ 16 MPI ranks x 4 OpenMP threads on 32-core x86; CLQCD configuration at m_s; precision not stated; "
                             "another machine and a thermalised configuration: context, not a target"}
    ctx.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--rows", default="all", help="'all', 'main' (skip the side measurements) or 'multi_rhs' (main + multi-rhs rows)")
    ap.add_argument("--nrhs", default="2,4,8", help="batch sizes of the multi-rhs rows")
    ap.add_argument("--batch-l2-bytes", type=float, default=None, help="override ddamg option batch_l2_bytes")
    ap.add_argument("--gauge-recon", type=int, default=12, choices=[18, 12],
                    help="link storage read by the fused hopping kernels: 18 reals, or two-row 12 reals (ddamg option gauge_recon)")
    args = ap.parse_args()
    global BYTES_A, BYTES_B, BYTES_BR
    if args.gauge_recon == 12:          # 8 links x (72 - 48) B less per output site and kernel
        BYTES_A, BYTES_B, BYTES_BR = BYTES_A - 192, BYTES_B - 192, BYTES_BR - 192
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    import torch.distributed as dist
    import gen
    from paper_2407_08092_b200 import Ddamg, F32, build_library

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    if rank == 0:
        build_library()
    if world > 1:
        dist.barrier()

    W, K = max(3, args.warmup), max(1, args.steps)
    cfg = args.config
    c = CONFIGS[cfg]
    L, T = c["L"], c["T"]
    V = L * L * L * T
    Ve = V // 2
    stream = torch.cuda.current_stream()

    def ev():
        return torch.cuda.Event(enable_timing=True)

    # ---- setup: a0, a1 (timed once, reported, not part of a step)
    ctx = Ddamg(L, T, c["csw"], c["m0"], c["bc"], F32, stream=None, device=dev)
    t0 = time.perf_counter()
    U = gen.gauge_field(L, T, 1000 + cfg, c["eps"], c["reunit"], device=dev, dtype=torch.complex64)
    torch.cuda.synchronize()
    t_gen = time.perf_counter() - t0
    e0, e1, e2 = ev(), ev(), ev()
    e0.record()
    ctx.load_gauge(U)
    e1.record()
    ctx.build_clover()
    e2.record()
    if args.gauge_recon == 12:
        ctx.set_option("gauge_recon", 12)
    torch.cuda.synchronize()
    t_a0, t_a1 = e0.elapsed_time(e1), e1.elapsed_time(e2)
    del U
    torch.cuda.empty_cache()

    # ---- inputs: a pool of Gaussian rhs / initial guesses, generated outside any timed region
    NPOOL = 3

    def fresh(seed):
        nat = gen.spinor_field(L, T, seed, device=dev, dtype=torch.complex64)
        xe, xo = ctx.pack(nat)
        torch.cuda.synchronize()
        del nat
        return xe, xo

    pool_b, pool_x = [], []
    for i in range(NPOOL):
        be, bo = fresh(2000 + cfg + i)
        pool_b.append((be, bo))
        pool_x.append(fresh(3000 + cfg + i)[0])
    x_e = ctx.half_spinor()
    y_e = ctx.half_spinor()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warm, prep=None):
        """Sum of per-step CUDA-event times over `steps` steps; prep() runs outside the events."""
        for i in range(warm):
            if prep:
                prep(i)
            fn(i)
        barrier()
        pairs = []
        for i in range(steps):
            if prep:
                prep(i)
            a, b = ev(), ev()
            a.record()
            fn(i)
            b.record()
            pairs.append((a, b))
        barrier()
        ms = sum(a.elapsed_time(b) for a, b in pairs)
        return max_over_ranks(ms, world, dev)

    # ---- the step: fused Richardson smoother nu = 4 (rows a2-a7)
    def prep_x(i):
        x_e.copy_(pool_x[i % NPOOL])

    def step(i):
        ctx.richardson(pool_b[i % NPOOL][0], x_e, NU, c["omega"])

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()                      # sampled from the warm-up on, so short runs still see load
        sampler.wait_ready()
    ctx.kernel_timing(True)
    for i in range(W):
        prep_x(i); step(i)
    torch.cuda.synchronize()
    ctx.kernel_time_ms(0, reset=True)
    launches0 = ctx.launch_count()
    wall0 = time.perf_counter()
    ms_total = timed(step, K, 0, prep_x)
    wall = time.perf_counter() - wall0
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    msA, nA = ctx.kernel_time_ms(0, reset=False)
    msB, nB = ctx.kernel_time_ms(1, reset=True)
    ctx.kernel_timing(False)
    ms_per_step = ms_total / K
    value = job_value(V, NU, world, ms_per_step)

    peak, peak_src = _peaks()
    tB = msB / max(nB, 1) * 1e-3
    tA = msA / max(nA, 1) * 1e-3
    ach_B = BYTES_BR * Ve / tB / 1e9
    ach_A = BYTES_A * Ve / tA / 1e9
    roofline = {"bound": "hbm", "kernel": "dslash_kernel<float, EPI_RICHARDSON> (kernel B')",
                "achieved": ach_B, "peak": peak, "unit": "GB/s", "frac": ach_B / peak,
                "traffic": NCU_TRAFFIC_BYTES[args.gauge_recon].get(cfg), "peak_source": peak_src,
                "bytes_per_launch": BYTES_BR * Ve, "avg_launch_ms": tB * 1e3, "launches_timed": nB,
                "other_kernels": [{"kernel": "dslash_kernel<float, EPI_CLOV_HOP> (kernel A)", "achieved": ach_A,
                                   "frac": ach_A / peak, "bytes_per_launch": BYTES_A * Ve, "avg_launch_ms": tA * 1e3,
                                   "launches_timed": nA}],
                "sweep_two_pass": {"bytes": (BYTES_A + BYTES_BR) * Ve, "achieved": (BYTES_A + BYTES_BR) * Ve * NU / (ms_per_step * 1e-3) / 1e9,
                                   "frac": (BYTES_A + BYTES_BR) * Ve * NU / (ms_per_step * 1e-3) / 1e9 / peak}}

    rows = {"a0_load_gauge_ms": t_a0, "a1_build_clover_ms": t_a1, "input_generation_s": t_gen}
    if args.rows == "all" and args.gauge_recon == 12:
        # ---- the same step on full 18-real links (two-pass model 1056 + 1248 B per even site)
        ctx.set_option("gauge_recon", 18)
        ks = max(3, min(K, 10))
        ms18 = timed(step, ks, 3, prep_x) / ks
        ctx.set_option("gauge_recon", 12)
        b18 = (BYTES_A + BYTES_BR + 2 * 192) * Ve * NU
        rows["richardson_links18"] = {"ms_per_step": ms18, "site_sweeps_per_s": job_value(V, NU, world, ms18),
                                      "GBps_two_pass_model": b18 / (ms18 * 1e-3) / 1e9,
                                      "frac_of_peak": b18 / (ms18 * 1e-3) / 1e9 / peak,
                                      "bytes_per_even_site_sweep": BYTES_A + BYTES_BR + 2 * 192}
    if args.rows == "all":
        # ---- Schur apply (BASELINE.json metric: GB/s and GFLOP/s, fp32)
        ks = max(3, min(K, 20))
        ms = timed(lambda i: ctx.apply_schur(pool_x[i % NPOOL], y_e), ks, 3) / ks
        gbs = (BYTES_A + BYTES_B) * Ve / (ms * 1e-3) / 1e9
        rows["schur_apply"] = {"ms": ms, "sites_per_s": V / (ms * 1e-3), "GBps_two_pass_model": gbs,
                               "frac_of_peak": gbs / peak,
                               "GFLOPps": (FLOP_PER_SITE * V + 24 * Ve) / (ms * 1e-3) / 1e9}
        # ---- whole odd-even smoother call, eq. 2 (a10): prepare_rhs + nu sweeps from 0 + reconstruct_odd
        bhat = ctx.half_spinor()
        x_o = ctx.half_spinor()

        def smoother(i):
            be, bo = pool_b[i % NPOOL]
            ctx.prepare_rhs(be, bo, bhat)
            ctx.richardson(bhat, x_e, NU, c["omega"], zero_init=True)
            ctx.reconstruct_odd(bo, x_e, x_o)
        km = max(3, min(K, 10))
        ms = timed(smoother, km, 2) / km
        rows["smoother_call_eq2"] = {"ms": ms, "note": "prepare_rhs + Richardson(nu=4, x0=0: first sweep has no apply) + reconstruct_odd"}
        del bhat, x_o
        # ---- GMRES(1, 10) (a8, a9)
        try:
            kg = 10
            ms = timed(lambda i: ctx.gmres_oe(pool_b[i % NPOOL][0], x_e, kg, 1, zero_init=True), 2, 1) / 2
            rows["gmres_1x10"] = {"ms": ms, "ms_per_arnoldi_step": ms / kg}
        except Exception as e:     # e.g. Krylov basis does not fit
            rows["gmres_1x10"] = {"error": str(e)}
        # ---- SAP(3,4) on 4^4 blocks (NEXT-3; the smoother of the paper's Tables 2 and 6)
        try:
            xs_e, xs_o = ctx.half_spinor(), ctx.half_spinor()
            ctx.kernel_timing(True)
            ctx.kernel_time_ms(6, reset=True)
            ksap = 3
            ms = timed(lambda i: ctx.sap(pool_b[i % NPOOL][0], pool_b[i % NPOOL][1], xs_e, xs_o, SAP_N, SAP_M,
                                         SAP_BLOCK, zero_init=False), ksap, 1,
                       lambda i: (xs_e.copy_(pool_x[i % NPOOL]), xs_o.copy_(pool_x[(i + 1) % NPOOL]))) / ksap
            ms5, n5 = ctx.kernel_time_ms(5, reset=False)
            ms6, n6 = ctx.kernel_time_ms(6, reset=True)
            ctx.kernel_timing(False)
            t6 = ms6 / max(n6, 1) * 1e-3
            # block kernel: per block site pair 2m+2 in-block hopping sums and 2m+2 6x6x2 products
            flop_blk = (2 * SAP_M + 2) * (SAP_HOP_FLOP + 504) * Ve / 2
            rows["sap_3x4_block4"] = {
                "ms_per_call": ms, "site_iterations_per_s": V * SAP_N / (ms * 1e-3),
                "block_kernel_ms": t6 * 1e3, "block_kernel_launches": n6,
                "residual_kernel_ms": ms5 / max(n5, 1), "residual_kernel_launches": n5,
                "block_kernel_GFLOPps": flop_blk / t6 / 1e9,
                "block_kernel_bound": "latency (8 warps/SM; fp32 FMA pipe ~28 % busy, profiles/r1d_ncu_full_sap.md)",
                "note": "SAP(n=3, m=4), 4^4 blocks, non-zero x0: per iteration and colour one streaming residual "
                        "(2 launches) + one block-solve launch"}
            del xs_e, xs_o
        except Exception as e:
            rows["sap_3x4_block4"] = {"error": str(e)}

    if args.rows in ("all", "multi_rhs"):
        # ---- multi-rhs batched Richardson (NEXT-2): links + clover fetched once for nrhs rhs
        rows["multi_rhs_richardson"] = {}
        if args.batch_l2_bytes is not None:
            ctx.set_option("batch_l2_bytes", args.batch_l2_bytes)
        for nrhs in [int(t) for t in args.nrhs.split(",") if t]:
            try:
                Bb = torch.randn(nrhs * 12 * V, dtype=torch.float32, device=dev)
                X0 = torch.randn(nrhs * 12 * V, dtype=torch.float32, device=dev)
                Xb = torch.empty_like(X0)
                ctx.kernel_timing(True)
                ctx.kernel_time_ms(3, reset=True)
                kb = max(3, min(K, 5))
                ms = timed(lambda i: ctx.richardson_batch(nrhs, Bb, Xb, NU, c["omega"]), kb, 2,
                           lambda i: Xb.copy_(X0)) / kb
                ms3, n3 = ctx.kernel_time_ms(3, reset=False)
                ms4, n4 = ctx.kernel_time_ms(4, reset=True)
                ctx.kernel_timing(False)
                lk = 384 if args.gauge_recon == 12 else 576          # 8 links per output site
                bA = 192 + (lk + 288) / nrhs     # per (site, rhs): x_e neighbours 96 + write 96 + (links + clover 288) / nrhs
                bB = 384 + (lk + 288) / nrhs     # t_o 96 + x_e 96 + b_e 96 + write 96 + (links + 288) / nrhs
                tA3, tB4 = ms3 / max(n3, 1) * 1e-3, ms4 / max(n4, 1) * 1e-3
                rows["multi_rhs_richardson"][str(nrhs)] = {
                    "ms_per_call": ms, "rhs_site_sweeps_per_s": V * NU * nrhs / (ms * 1e-3),
                    "speedup_vs_single_rhs": (V * NU * nrhs / (ms * 1e-3)) / (V * NU / (ms_per_step * 1e-3)),
                    "kernel_A_ms": tA3 * 1e3, "kernel_A_model_GBps": bA * nrhs * Ve / tA3 / 1e9,
                    "kernel_Bp_ms": tB4 * 1e3, "kernel_Bp_model_GBps": bB * nrhs * Ve / tB4 / 1e9,
                    "model_bytes_per_rhs_site_sweep": bA + bB}
                del Bb, X0, Xb
                torch.cuda.empty_cache()
            except Exception as e:
                rows["multi_rhs_richardson"][str(nrhs)] = {"error": str(e)}

    if args.rows == "all" and rank == 0 and world == 1:
        # ---- context row: the paper's three smoother configurations (Table 2) on the
        # paper's lattice SHAPE 48^3 x 96 (synthetic links, fp32; the paper: CLQCD configuration, 16 GPUs
        # of 64 SMs / 16 GB HBM2 on 4 ORISE nodes, 32-core x86 hosts, precision not stated).  Context only.
        try:
            rows["paper_smoother_calls_48x96"] = paper_context_row(torch, gen, Ddamg, F32, dev, args.gauge_recon)
        except Exception as exc:                  # noqa: BLE001 - a side row must not lose the headline
            rows["paper_smoother_calls_48x96"] = {"error": str(exc)[:200]}
        try:
            rows["schur_apply_f64_48x96"] = f64_apply_row(torch, gen, Ddamg, dev)
        except Exception as exc:                  # noqa: BLE001
            rows["schur_apply_f64_48x96"] = {"error": str(exc)[:200]}

    # ---- e2e: HOST buffers, copies inside the timed region, through the public API
    hb = torch.empty_like(pool_b[0][0], device="cpu").pin_memory()
    hx = torch.empty_like(hb).pin_memory()
    hout = torch.empty_like(hb).pin_memory()
    hb.copy_(pool_b[0][0]); hx.copy_(pool_x[0])
    d_b = ctx.half_spinor()

    # Steps are independent, so the copies of neighbouring steps are pipelined: H2D of step i+1 and
    # D2H of step i-1 run on two copy streams while step i computes (double-buffered device inputs);
    # every step still moves its own inputs host->device and its own result device->host.
    d_b2, d_x2 = [d_b, ctx.half_spinor()], [x_e, ctx.half_spinor()]
    s_in, s_out = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    main = torch.cuda.current_stream()

    def e2e_run(nsteps):
        t0, t1 = ev(), ev()
        t0.record(main)
        s_in.wait_event(t0)
        freed = [None, None]
        last_out = None
        for i in range(nsteps):
            k = i & 1
            with torch.cuda.stream(s_in):
                if freed[k] is not None:
                    s_in.wait_event(freed[k])                 # buffer k was read back by step i-2
                d_b2[k].copy_(hb, non_blocking=True)
                d_x2[k].copy_(hx, non_blocking=True)
                e_in = ev(); e_in.record(s_in)
            main.wait_event(e_in)
            ctx.richardson(d_b2[k], d_x2[k], NU, c["omega"])
            e_done = ev(); e_done.record(main)
            with torch.cuda.stream(s_out):
                s_out.wait_event(e_done)
                hout.copy_(d_x2[k], non_blocking=True)
                freed[k] = ev(); freed[k].record(s_out)
                last_out = freed[k]
        main.wait_event(last_out)
        t1.record(main)
        return t0, t1
    ke = max(3, min(K, 10))
    e2e_run(2)
    barrier()
    t0, t1 = e2e_run(ke)
    barrier()
    ms_e2e = max_over_ranks(t0.elapsed_time(t1), world, dev) / ke
    e2e = {"value": job_value(V, NU, world, ms_e2e), "unit": "site-sweeps/s", "ms_per_step": ms_e2e,
           "h2d_bytes_per_step": 2 * ctx.half_bytes, "d2h_bytes_per_step": ctx.half_bytes,
           "note": "through Ddamg.richardson with pinned HOST buffers; per step H2D of b_e and x0, the call, D2H of x^(nu); "
                   "copies of neighbouring steps overlap the compute (two copy streams, double-buffered inputs)"}

    line = {
        "metric": "Richardson sites/s (odd-even Schur Wilson-clover, nu=4)",
        "value": value, "unit": "site-sweeps/s", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config {cfg}: {L}^3x{T} lattice ({V} sites), Wilson-clover csw={c['csw']} m0={c['m0']}, "
                               f"links exp(i*{c['eps']}*H) reunitarised, antiperiodic t; step = ddamg_richardson(nu={NU}, "
                               f"omega={c['omega']}) on Gaussian b_e and non-zero Gaussian x0",
                   "l2_policy": "working set per sweep (gauge+clover+spinors = %.1f GB) is far larger than the 126 MB L2; no flush needed"
                                % ((BYTES_A + BYTES_BR) * Ve / 1e9),
                   "gauge_recon": args.gauge_recon,
                   "bytes_per_even_site": {"kernel_A": BYTES_A, "kernel_B": BYTES_B, "kernel_Bprime": BYTES_BR},
                   "multi_gpu": "replicas only (no sharding, no collective on the data path)",
                   "timing": "sum of per-step CUDA-event times on the launching stream; x0 refresh copy outside the events",
                   "wall_s_timed_region": wall},
        "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "rows": rows,
    }
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            r = oracle_run(6, 1, cfg)
            line["cpu_baseline"] = {"value": r["value"], "unit": "site-sweeps/s", "cores": r["cores"],
                                    "kind": "oracle", "sample": r["sample"]}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
