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
             1184 B/even site (18-real links; 992 B with two-row links) / CUDA-event duration,
             against MEASURED_PEAKS.json
cpu_baseline = the fp64 oracle (oracle/, as it stands) timed on the host cores on a bounded
             sample (16^3 x 32 lattice, same recipe: `value`), plus SURVEY.md 8(d)'s table: Schur
             apply and one Richardson sweep at 16^4 and 32^3 x 64, all cores and 1 thread, with the
             CPU model string
--rows     = 'all' (default), 'main' (the step only) or a comma list of side rows:
             links18,schur,smoother,gmres,gcr,sap,multi_rhs,paper,f64,cfg2,cfg3,cfg4
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
CLOV_A = 224            # A_ee in the compact 28-real form (2 x 28 x 4 B; SURVEY.md's model has the packed 288 B)
BYTES_A = 1056          # kernel A : 8 links 576 + x_e neighbours 96 + A_oo^-1 288 + write 96
BYTES_B = 864 + CLOV_A  # kernel B : 8 links 576 + t_o 96 + x_e 96 + A_ee 224 + write 96  (= 1088; 1152)
BYTES_BR = BYTES_B + 96 # kernel B': kernel B + b_e 96                                     (= 1184; 1248)
FLOP_PER_SITE = 1824    # 1320 (hop) + 504 (2 x 6x6 Hermitian mat-vec), per lattice site
# dram__bytes_read.sum + dram__bytes_write.sum per launch of kernel B' at config 5, from the
# ncu --set full capture summarised in profiles/ (None until a capture exists)
NCU_TRAFFIC_BYTES = {18: {5: 20.194e9}, 12: {5: 16.956e9}}     # profiles/r2b_ncu_full_dslash18.md, profiles/r2b_ncu_full_dslash12.md
NOMINAL_HBM_GBS = 8000.0    # north_star's "~8 TB/s HBM peak" (DGX figure; HGX 7.7 TB/s), quoted beside the measured copy peak
SIDE_ROWS = ("links18", "schur", "smoother", "gmres", "gcr", "sap", "multi_rhs", "paper", "f64", "cfg2", "cfg3", "cfg4")
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


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def oracle_detail(cfg: int, device=None):
    """SURVEY.md 8(d) "Oracle timing beside it": the oracle's Schur apply and ONE Richardson sweep at 16^4 and
    32^3 x 64 (recipe of `cfg`), with all host cores and with 1 thread.  Inputs are generated outside the
    timed calls (on `device` when given); the oracle itself runs as it stands (OpenMP over sites, numpy axpy)."""
    import ctypes
    import numpy as np
    import gen
    import oracle
    c = CONFIGS[cfg]
    ncores = os.cpu_count() or 1
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
    except OSError:
        gomp = None
    out = {}
    for L, T, tag in ((16, 16, "16x16"), (32, 64, "32x64")):
        kw = dict(device=device) if device is not None else {}
        U = gen.gauge_field(L, T, 1000 + cfg, c["eps"], c["reunit"], **kw).cpu().numpy()
        op = oracle.WilsonClover(L, T, c["csw"], c["m0"], c["bc"], U)
        b = np.where(op.even, gen.spinor_field(L, T, 2000 + cfg, **kw).cpu().numpy(), 0.0)
        x0 = np.where(op.even, gen.spinor_field(L, T, 2500 + cfg, **kw).cpu().numpy(), 0.0)
        V = L * L * L * T
        for nt, name in ((ncores, "allcores"), (1, "1thread")):
            if gomp is None and nt != ncores:
                continue
            if gomp is not None:
                gomp.omp_set_num_threads(nt)
            reps = 2 if (nt > 1 or V < 1 << 20) else 1
            op.apply_schur(x0)                                    # warm-up (page-in)
            t0 = time.perf_counter()
            for _ in range(reps):
                op.apply_schur(x0)
            ta = (time.perf_counter() - t0) / reps
            t0 = time.perf_counter()
            for _ in range(reps):
                oracle.richardson(op.apply_schur, b, x0, 1, c["omega"])
            ts = (time.perf_counter() - t0) / reps
            out[f"schur_apply_{tag}_{name}_sites_per_s"] = V / ta
            out[f"richardson_sweep_{tag}_{name}_sites_per_s"] = V / ts
        if gomp is not None:
            gomp.omp_set_num_threads(ncores)
        del op, U, b, x0
    out["threads_allcores"] = ncores
    return out


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
                         "sample": r["sample"], "cpu_model": cpu_model()},
        "e2e": {"value": r["value"], "unit": "site-sweeps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------- our arm
def f64_apply_row(torch, gen, Ddamg, dev):
    """fp64 Schur apply at 48^3 x 96 (config 4 recipe, 18-real links): the precision of BASELINE.json's
    fp64 parity bar, timed against the two-pass byte model at 8 bytes per real (2 x (1056 + 1088) = 4288 B per even site)."""
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
    gbs = 2 * (1056 + 864 + CLOV_A) * (V // 2) / (ms * 1e-3) / 1e9     # 18-real links, whatever --gauge-recon says
    ctx.close()
    return {"lattice": "48^3x96, fp64, 18-real links", "ms": ms, "sites_per_s": V / (ms * 1e-3),
            "GBps_two_pass_model": gbs, "frac_of_peak": gbs / peak,
            "GFLOPps": (FLOP_PER_SITE * V + 24 * (V // 2)) / (ms * 1e-3) / 1e9}


def config4_rows(torch, gen, Ddamg, F32, dev, recon, want_paper, gmres_split):
    """Rows on the 48^3 x 96 lattice (BASELINE.json configs[3] = the paper's lattice shape): (i) one smoother call
    each of odd-even Richardson(12, 1.5), odd-even GMRES(3, 4) and SAP(3, 4) beside the paper's Table 2; (ii) config 4
    as written: odd-even GMRES(2, 10) from x0 = 0 on a Gaussian rhs, time per Arnoldi step split apply / BLAS-1."""
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
    bhat, x_e, x_o = ctx.half_spinor(), ctx.half_spinor(), ctx.half_spinor()
    res = {}
    if gmres_split is not None:
        ctx.prepare_rhs(b_e, b_o, bhat)
        g = gmres_split(ctx, bhat, x_e, 10, 2, L * L * L * T, 3)
        g["lattice"] = "48^3x96, fp32, GMRES(n=2, m=10) from x0=0: 20 Arnoldi steps + 3 residual evaluations"
        res["gmres_2x10_cfg4"] = g
    if not want_paper:
        ctx.close()
        return res
    v = b_e.clone()
    lam = ctx.power_iteration(v, 10)              # Alg. 4 line 1: omega = delta / |lambda_max|, delta = 1.5
    omega = 1.5 / lam

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

    res["paper_smoother_calls_48x96"] = {
           "lattice": "48^3x96 (the paper's 96x48^3 shape), synthetic links, fp32, one B200",
           "omega_power_iteration": omega,
           "odd_even_richardson_12_ms": timed_call(rich), "odd_even_gmres_3x4_ms": timed_call(gm),
           "sap_3x4_ms": timed_call(sap),
           "paper_gpu_ms": {"odd_even_richardson": 360.0, "odd_even_gmres_3x4": 450.0, "sap_3x4": 330.0},
           "paper_cpu_ms": {"odd_even_richardson": 4800.0, "odd_even_gmres_3x4": 5660.0, "sap_3x4": 4390.0},
           "paper_hardware": "Table 2, PAPER.md:258-262: 4 ORISE nodes, 16 GPUs (64 SMs, 16 GB HBM2, HIP, host-staged halos) "
                             "/ 16 MPI ranks x 4 OpenMP threads on 32-core x86; CLQCD configuration at m_s; precision not stated; "
                             "another machine and a thermalised configuration: context, not a target"}
    ctx.close()
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=sorted(CONFIGS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--rows", default="all", help="'all', 'main' (the step only) or a comma list of side rows: " + ",".join(SIDE_ROWS))
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
    sel = set(SIDE_ROWS) if args.rows == "all" else set() if args.rows == "main" else {t for t in args.rows.split(",") if t}
    unknown = sel - set(SIDE_ROWS)
    assert not unknown, f"unknown --rows entries {sorted(unknown)}; known: {SIDE_ROWS}"
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

    def step_stats(per):
        q = sorted(per)
        return {"median": q[len(q) // 2] if len(q) % 2 else 0.5 * (q[len(q) // 2 - 1] + q[len(q) // 2]), "min": q[0],
                "p95": q[min(len(q) - 1, int(0.95 * len(q)))], "max": q[-1], "n": len(q)}

    last_per_step = []

    def timed(fn, steps, warm, prep=None):
        """Sum of per-step CUDA-event times over `steps` steps; prep() runs outside the events.
        The per-step times of the last call stay in last_per_step (this rank's)."""
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
        last_per_step[:] = [a.elapsed_time(b) for a, b in pairs]
        ms = sum(last_per_step)
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
    stats = step_stats(last_per_step)
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
    sweep_gbs = (BYTES_A + BYTES_BR) * Ve * NU / (ms_per_step * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "dslash_kernel<float, EPI_RICHARDSON> (kernel B')",
                "achieved": ach_B, "peak": peak, "unit": "GB/s", "frac": ach_B / peak,
                "traffic": NCU_TRAFFIC_BYTES[args.gauge_recon].get(cfg), "peak_source": peak_src,
                "traffic_source": "ncu --set full capture of one launch, profiles/ (a citation, not re-measured by this run)"
                                  if NCU_TRAFFIC_BYTES[args.gauge_recon].get(cfg) else None,
                "bytes_per_launch": BYTES_BR * Ve, "avg_launch_ms": tB * 1e3, "launches_timed": nB,
                # flat copies of the other hot kernel and of the whole step (nested objects may be cut by a parser)
                "kernel_A_achieved": ach_A, "kernel_A_frac": ach_A / peak, "kernel_A_avg_launch_ms": tA * 1e3,
                "kernel_A_bytes_per_launch": BYTES_A * Ve,
                "sweep_two_pass_achieved": sweep_gbs, "sweep_two_pass_frac": sweep_gbs / peak,
                "frac_of_nominal_8TBps": ach_B / NOMINAL_HBM_GBS, "kernel_A_frac_of_nominal_8TBps": ach_A / NOMINAL_HBM_GBS,
                "sweep_frac_of_nominal_8TBps": sweep_gbs / NOMINAL_HBM_GBS,
                "peak_note": "the measured peak is a 50/50 read/write copy; these kernels are >= 90 % reads, and a read-dominated "
                             "stream runs a few % above a copy on HBM3e, so a frac slightly above 1 is a peak-calibration artefact, "
                             "not extra work: ncu DRAM traffic = 1.02 x algorithmic bytes (profiles/)",
                "other_kernels": [{"kernel": "dslash_kernel<float, EPI_CLOV_HOP> (kernel A)", "achieved": ach_A,
                                   "frac": ach_A / peak, "bytes_per_launch": BYTES_A * Ve, "avg_launch_ms": tA * 1e3,
                                   "launches_timed": nA}],
                "sweep_two_pass": {"bytes": (BYTES_A + BYTES_BR) * Ve, "achieved": (BYTES_A + BYTES_BR) * Ve * NU / (ms_per_step * 1e-3) / 1e9,
                                   "frac": (BYTES_A + BYTES_BR) * Ve * NU / (ms_per_step * 1e-3) / 1e9 / peak}}

    rows = {"a0_load_gauge_ms": t_a0, "a1_build_clover_ms": t_a1, "input_generation_s": t_gen}
    flat = {}        # scalar copies of side-row results for the `config` object (nested rows may be cut by a parser)

    def gmres_split(cx, be, xe, k, cycles, Vloc, reps):
        """One odd-even GMRES(cycles, k) call: total time and its split into operator applications (kernel
        classes A, B) and BLAS-1 passes (classes multi-dot, multi-axpy, other streaming passes), CUDA events
        recorded by the library around every launch."""
        cx.gmres_oe(be, xe, k, cycles, zero_init=True)                       # warm-up (allocates the basis)
        cx.kernel_timing(True)
        cx.kernel_time_ms(0, reset=True)
        ms = timed(lambda i: cx.gmres_oe(be, xe, k, cycles, zero_init=True), reps, 0) / reps
        t = {w: cx.kernel_time_ms(w, reset=False) for w in (0, 1, 8, 9, 10)}
        cx.kernel_time_ms(0, reset=True)
        cx.kernel_timing(False)
        steps_ = k * cycles * reps
        apply_ms = (t[0][0] + t[1][0]) / steps_
        vb = 96 * (Vloc // 2)                                                # bytes of one half spinor
        nb_dot = sum(j + 2 for j in range(k)) * cycles * reps                # vectors read by the multi-dots
        nb_axpy = (sum(j + 3 for j in range(k)) + (k + 2)) * cycles * reps   # read + written by the multi-axpys (+ x += V y)
        out = {"ms": ms, "ms_per_arnoldi_step": ms / (k * cycles),
               "apply_ms_per_arnoldi_step": apply_ms,
               "blas1_ms_per_arnoldi_step": (t[8][0] + t[9][0] + t[10][0]) / steps_,
               "multi_dot_ms_per_arnoldi_step": t[8][0] / steps_, "multi_axpy_ms_per_arnoldi_step": t[9][0] / steps_,
               "other_blas1_ms_per_arnoldi_step": t[10][0] / steps_,
               "multi_dot_GBps": nb_dot * vb / (t[8][0] * 1e-3) / 1e9 if t[8][0] > 0 else None,
               "multi_axpy_GBps": nb_axpy * vb / (t[9][0] * 1e-3) / 1e9 if t[9][0] > 0 else None,
               "note": "apply = kernels A + B (incl. the residuals at cycle start / end); blas1 = fused multi-dot, "
                       "multi-axpy + norm and copy passes; remainder = small device-side scalar kernels and launch gaps"}
        if out["multi_dot_GBps"]:
            out["multi_dot_frac_of_peak"] = out["multi_dot_GBps"] / peak
            out["multi_axpy_frac_of_peak"] = out["multi_axpy_GBps"] / peak
        return out

    if "links18" in sel and args.gauge_recon == 12:
        # ---- the same step on full 18-real links (two-pass model 1056 + 1184 B per even site)
        ctx.set_option("gauge_recon", 18)
        ks = max(3, min(K, 10))
        ms18 = timed(step, ks, 3, prep_x) / ks
        ctx.set_option("gauge_recon", 12)
        b18 = (BYTES_A + BYTES_BR + 2 * 192) * Ve * NU
        rows["richardson_links18"] = {"ms_per_step": ms18, "site_sweeps_per_s": job_value(V, NU, world, ms18),
                                      "GBps_two_pass_model": b18 / (ms18 * 1e-3) / 1e9,
                                      "frac_of_peak": b18 / (ms18 * 1e-3) / 1e9 / peak,
                                      "bytes_per_even_site_sweep": BYTES_A + BYTES_BR + 2 * 192}
        flat["links18_ms_per_step"] = ms18
        flat["links18_frac_of_peak"] = rows["richardson_links18"]["frac_of_peak"]
    if "schur" in sel:
        # ---- Schur apply (BASELINE.json metric: GB/s and GFLOP/s, fp32)
        ks = max(3, min(K, 20))
        ms = timed(lambda i: ctx.apply_schur(pool_x[i % NPOOL], y_e), ks, 3) / ks
        gbs = (BYTES_A + BYTES_B) * Ve / (ms * 1e-3) / 1e9
        rows["schur_apply"] = {"ms": ms, "sites_per_s": V / (ms * 1e-3), "GBps_two_pass_model": gbs,
                               "frac_of_peak": gbs / peak, "frac_of_nominal_8TBps": gbs / NOMINAL_HBM_GBS,
                               "GFLOPps": (FLOP_PER_SITE * V + 24 * Ve) / (ms * 1e-3) / 1e9,
                               "per_call_ms": step_stats(last_per_step)}
        flat.update(schur_apply_ms=ms, schur_apply_GBps=gbs, schur_apply_GFLOPps=rows["schur_apply"]["GFLOPps"],
                    schur_apply_frac_of_peak=gbs / peak)
    if "smoother" in sel:
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
    if "gmres" in sel:
        # ---- GMRES(1, 10) (a8, a9) at the bench lattice, split into apply / BLAS-1
        try:
            rows["gmres_1x10"] = gmres_split(ctx, pool_b[0][0], x_e, 10, 1, V, 2)
            flat.update(gmres_1x10_ms_per_arnoldi_step=rows["gmres_1x10"]["ms_per_arnoldi_step"],
                        gmres_1x10_multi_dot_frac_of_peak=rows["gmres_1x10"].get("multi_dot_frac_of_peak"),
                        gmres_1x10_multi_axpy_frac_of_peak=rows["gmres_1x10"].get("multi_axpy_frac_of_peak"))
        except Exception as e:     # e.g. Krylov basis does not fit
            rows["gmres_1x10"] = {"error": str(e)}
    if "gcr" in sel:
        # ---- GCR(1, 10) (NEXT-4, Alg. 3): same operator applications as GMRES, fused form / update passes
        try:
            ctx.gcr_oe(pool_b[0][0], x_e, 10, 1, zero_init=True)           # warm-up (allocates the 2k + 1 vectors)
            ctx.kernel_timing(True)
            ctx.kernel_time_ms(0, reset=True)
            ms = timed(lambda i: ctx.gcr_oe(pool_b[0][0], x_e, 10, 1, zero_init=True), 2, 0) / 2
            tk = {w: ctx.kernel_time_ms(w, reset=False)[0] for w in (0, 1, 8, 10)}
            ctx.kernel_time_ms(0, reset=True)
            ctx.kernel_timing(False)
            rows["gcr_1x10"] = {"ms": ms, "ms_per_step": ms / 10, "apply_ms_per_step": (tk[0] + tk[1]) / 20,
                                "blas1_ms_per_step": (tk[8] + tk[10]) / 20,
                                "note": "blas1 = multi-dot against the z_j + fused form pass (z, p, next delta) + update pass"}
            flat["gcr_1x10_ms_per_step"] = ms / 10
        except Exception as e:
            rows["gcr_1x10"] = {"error": str(e)[:200]}
    if "sap" in sel:
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
                "note": "SAP(n=3, m=4), 4^4 blocks, non-zero x0"}
            flat["sap_3x4_ms_per_call"] = ms
            del xs_e, xs_o
        except Exception as e:
            rows["sap_3x4_block4"] = {"error": str(e)}

    if "multi_rhs" in sel:
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
                bB = 384 + (lk + CLOV_A) / nrhs  # t_o 96 + x_e 96 + b_e 96 + write 96 + (links + compact A_ee 224) / nrhs
                tA3, tB4 = ms3 / max(n3, 1) * 1e-3, ms4 / max(n4, 1) * 1e-3
                rate = V * NU * nrhs / (ms * 1e-3)
                rows["multi_rhs_richardson"][str(nrhs)] = {
                    "ms_per_call": ms, "rhs_site_sweeps_per_s": rate,
                    "speedup_vs_single_rhs": rate / (V * NU / (ms_per_step * 1e-3)),
                    "kernel_A_ms": tA3 * 1e3, "kernel_A_model_GBps": bA * nrhs * Ve / tA3 / 1e9,
                    "kernel_Bp_ms": tB4 * 1e3, "kernel_Bp_model_GBps": bB * nrhs * Ve / tB4 / 1e9,
                    "model_bytes_per_rhs_site_sweep": bA + bB,
                    "frac_of_byte_model": (bA + bB) * Ve * rate / V / 1e9 / peak}
                flat[f"multi_rhs_{nrhs}_rhs_site_sweeps_per_s"] = rate
                flat[f"multi_rhs_{nrhs}_frac_of_byte_model"] = rows["multi_rhs_richardson"][str(nrhs)]["frac_of_byte_model"]
                del Bb, X0, Xb
                torch.cuda.empty_cache()
            except Exception as e:
                rows["multi_rhs_richardson"][str(nrhs)] = {"error": str(e)}

    if "cfg2" in sel and rank == 0 and world == 1:
        # ---- BASELINE.json configs[1] (SURVEY.md 8(d) cfg 2): 16^4, 8 sweeps omega=1.0.  Gauge + clover = 38 MB << L2:
        # an L2-resident, launch-bound timing, NOT an HBM measurement; reported with and without the CUDA-graph
        # replay of the 2 nu launches of a history-free call (option "cuda_graph")
        try:
            c2 = CONFIGS[2]
            L2, T2 = c2["L"], c2["T"]
            V2 = L2 ** 3 * T2
            ctx2 = Ddamg(L2, T2, c2["csw"], c2["m0"], c2["bc"], F32, stream=None, device=dev)
            ctx2.load_gauge(gen.gauge_field(L2, T2, 1002, c2["eps"], c2["reunit"], device=dev, dtype=torch.complex64))
            ctx2.build_clover()
            b2 = ctx2.pack(gen.spinor_field(L2, T2, 2002, device=dev, dtype=torch.complex64), want_odd=False)[0]
            x2 = ctx2.half_spinor()
            row2 = {"lattice": "16^4 (fp32, 18-real links)", "nu": 8,
                    "note": "L2-resident (gauge + clover 38 MB): launch-bound, not an HBM measurement; 40 calls each (CUDA events per call), x0 = 0"}
            for name, mode in (("launches", 0), ("cuda_graph", 1)):
                ctx2.set_option("cuda_graph", mode)
                timed(lambda i: ctx2.richardson(b2, x2, 8, c2["omega"], zero_init=True), 40, 5)
                st2 = step_stats(last_per_step)
                row2[name + "_us_per_call"] = {k: (v * 1e3 if k != "n" else v) for k, v in st2.items()}
                flat[f"cfg2_{name}_us_per_call_median"] = st2["median"] * 1e3
            row2["site_sweeps_per_s_cuda_graph_median"] = V2 * 8 / (row2["cuda_graph_us_per_call"]["median"] * 1e-6)
            rows["config2_richardson_8_sweeps"] = row2
            ctx2.close()
            del ctx2, b2, x2
        except Exception as exc:                  # noqa: BLE001
            rows["config2_richardson_8_sweeps"] = {"error": str(exc)[:200]}

    if "cfg3" in sel and rank == 0 and world == 1:
        # ---- BASELINE.json configs[2] as written (SURVEY.md 8(d) cfg 3): 32^3 x 64, 100 calls of Richardson nu=4
        # omega=0.9, each on a FRESH Gaussian b_e and non-zero Gaussian x0 (generated outside the events),
        # 10 warm-up calls; per-call median / min / p95.  Gauge + clover (2 x 0.4 GB two-row / 0.6 GB) >> L2.
        try:
            c3 = CONFIGS[3]
            L3, T3 = c3["L"], c3["T"]
            V3 = L3 ** 3 * T3
            ctx3 = Ddamg(L3, T3, c3["csw"], c3["m0"], c3["bc"], F32, stream=None, device=dev)
            ctx3.load_gauge(gen.gauge_field(L3, T3, 1003, c3["eps"], c3["reunit"], device=dev, dtype=torch.complex64))
            ctx3.build_clover()
            if args.gauge_recon == 12:
                ctx3.set_option("gauge_recon", 12)
            b3, x3 = ctx3.half_spinor(), ctx3.half_spinor()

            def fresh3(i):
                b3.copy_(ctx3.pack(gen.spinor_field(L3, T3, 2003 + i, device=dev, dtype=torch.complex64), want_odd=False)[0])
                x3.copy_(ctx3.pack(gen.spinor_field(L3, T3, 3003 + i, device=dev, dtype=torch.complex64), want_odd=False)[0])
            ms = timed(lambda i: ctx3.richardson(b3, x3, NU, c3["omega"]), 100, 10, fresh3) / 100
            st3 = step_stats(last_per_step)
            rows["config3_richardson_100_calls"] = {
                "lattice": "32^3x64", "ms_per_call_mean": ms, "per_call_ms": st3,
                "site_sweeps_per_s_median": V3 * NU / (st3["median"] * 1e-3),
                "GBps_two_pass_model_median": (BYTES_A + BYTES_BR) * (V3 // 2) * NU / (st3["median"] * 1e-3) / 1e9,
                "note": "100 calls, fresh Gaussian b_e and x0 per call, 10 warm-up calls"}
            flat.update(cfg3_call_ms_median=st3["median"], cfg3_call_ms_min=st3["min"], cfg3_call_ms_p95=st3["p95"])
            ctx3.close()
            del ctx3, b3, x3
            torch.cuda.empty_cache()
        except Exception as exc:                  # noqa: BLE001 - a side row must not lose the headline
            rows["config3_richardson_100_calls"] = {"error": str(exc)[:200]}

    if ("paper" in sel or "cfg4" in sel) and rank == 0 and world == 1:
        # ---- 48^3 x 96 (BASELINE.json configs[3]; also the paper's lattice shape, Table 5)
        try:
            res4 = config4_rows(torch, gen, Ddamg, F32, dev, args.gauge_recon, "paper" in sel,
                                gmres_split if "cfg4" in sel else None)
            rows.update(res4)
            g4 = res4.get("gmres_2x10_cfg4")
            if g4 and "ms" in g4:
                flat.update(cfg4_gmres_2x10_ms=g4["ms"], cfg4_ms_per_arnoldi_step=g4["ms_per_arnoldi_step"],
                            cfg4_apply_ms_per_arnoldi_step=g4["apply_ms_per_arnoldi_step"],
                            cfg4_blas1_ms_per_arnoldi_step=g4["blas1_ms_per_arnoldi_step"])
        except Exception as exc:                  # noqa: BLE001
            rows["paper_smoother_calls_48x96"] = {"error": str(exc)[:200]}
    if "f64" in sel and rank == 0 and world == 1:
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

    if "smoother" in sel and rank == 0 and world == 1:
        # ---- what a caller with NATURAL-layout host fields pays for one whole smoother call (eq. 2): H2D of the
        # full-lattice rhs b (T,L,L,L,4,3 complex64), pack, prepare_rhs, Richardson(nu=4) from x0 = 0,
        # reconstruct_odd, unpack, D2H of the full-lattice x -- serial, one call after the other
        try:
            del hb, hx, hout
            nat_shape = (T, L, L, L, 4, 3)
            h_b = torch.empty(nat_shape, dtype=torch.complex64).pin_memory()
            h_x = torch.empty(nat_shape, dtype=torch.complex64).pin_memory()
            h_b.copy_(ctx.unpack(pool_b[0][0], pool_b[0][1]))
            d_nat = torch.empty(nat_shape, dtype=torch.complex64, device=dev)
            bhat, xo_ = ctx.half_spinor(), ctx.half_spinor()

            def natural_call(i):
                d_nat.copy_(h_b, non_blocking=True)
                be_, bo_ = ctx.pack(d_nat)
                ctx.prepare_rhs(be_, bo_, bhat)
                ctx.richardson(bhat, x_e, NU, c["omega"], zero_init=True)
                ctx.reconstruct_odd(bo_, x_e, xo_)
                h_x.copy_(ctx.unpack(x_e, xo_), non_blocking=True)
            kn = 3
            ms = timed(natural_call, kn, 1) / kn
            rows["e2e_smoother_call_natural_layout"] = {
                "ms": ms, "h2d_bytes": h_b.numel() * 8, "d2h_bytes": h_x.numel() * 8,
                "note": "host natural layout -> H2D -> pack -> eq.-2 smoother call (nu=4, x0=0) -> unpack -> D2H, serial; "
                        "PCIe-bound: 3.2 GB in + 3.2 GB out"}
            flat["e2e_smoother_call_natural_ms"] = ms
            del h_b, h_x, d_nat, bhat, xo_
        except Exception as exc:                  # noqa: BLE001
            rows["e2e_smoother_call_natural_layout"] = {"error": str(exc)[:200]}

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
                   "wall_s_timed_region": wall,
                   "step_ms_median": stats["median"], "step_ms_min": stats["min"], "step_ms_p95": stats["p95"]},
        "ms_per_step_median": stats["median"], "ms_per_step_min": stats["min"], "ms_per_step_p95": stats["p95"],
        "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "rows": rows,
    }
    line["config"].update({k: v for k, v in flat.items() if v is not None})
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            r = oracle_run(6, 1, cfg)
            line["cpu_baseline"] = {"value": r["value"], "unit": "site-sweeps/s", "cores": r["cores"],
                                    "kind": "oracle", "sample": r["sample"], "cpu_model": cpu_model()}
            try:            # apply and one sweep at 16^4 and 32^3x64, all cores and 1 thread
                line["cpu_baseline"].update(oracle_detail(cfg, dev))
            except Exception as exc:      # noqa: BLE001
                line["cpu_baseline"]["detail_error"] = str(exc)[:200]
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
