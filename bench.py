#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arxiv/paper_1009_5169 on B200.

A "step" is one MD force evaluation (Algorithm 2): the blocked mixed-precision solve
D X = Phi, the blocked solve D^dag Y = X (both to a true fp64 relative residual of 1e-12) and the
force accumulation F += sum_i f[x_i, y_i], over all n_rhs pseudo-fermion fields, all in the CUDA
kernels of libwd.so through its C ABI (inner fp32 links: 18 reals by default, --recon 12 for the compressed
form).  Workload at N = 1: BASELINE.json configs[4] at n_rhs = 5
(24^3 x 24 SF lattice, eps 0.4, kappa 0.135) -- the largest single-GPU config and the only one whose
working set (about 0.65 GB of solver vectors + 96 MB of fp32 links) is far outside the 126 MB L2,
so no L2 flush is needed between steps.  N > 1: independent replicas (the path has no exchange step,
DESIGN.md "Multi-GPU"), weak scaling.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--n-rhs 5] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "md_force_evals_per_s (2 blocked mixed-precision solves to 1e-12 + force; ms_per_step = solve time per MD force)"
UNIT = "force_eval/s"
TOL = 1e-12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="index into BASELINE.json configs")
    ap.add_argument("--n-rhs", type=int, default=5)
    ap.add_argument("--recon", type=int, default=18, choices=(12, 18), help="inner fp32 link form")
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--hop-impl", type=int, default=-1, choices=(-1, 0, 1, 2, 3),
                    help="WD_OPT_HOP_IMPL: 0 register kernel, 1 row-group ring kernel, 2 z-march or ring by shape (library default), "
                         "3 z-march wherever it runs, -1 leave the default")
    # the two tables BASELINE.json's configs[3] and configs[4] ask for are part of the default line (about 20 s); --quick
    # leaves them out.  --rhs-sweep / --apply-sweep are still accepted (they were the opt-in switches of earlier rounds).
    ap.add_argument("--quick", action="store_true", help="skip the configs[4] n_rhs sweep and the configs[3] 16^4 apply table")
    ap.add_argument("--rhs-sweep", action="store_true", help="(default on) configs[4]: blocked solve at n_rhs = 1, 2, 5, 8, 12")
    ap.add_argument("--apply-sweep", action="store_true", help="(default on) configs[3]: D, D^dag apply on 16^4, fp32/fp64 x 18/12 reals")
    ap.add_argument("--shard-rhs", action="store_true",
                    help="N > 1: deal the n_rhs columns of ONE problem to the ranks (gauge replicated, allReduce of F): strong scaling")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-baseline-full", action="store_true", help="time the oracle on the WHOLE workload (minutes)")
    ap.add_argument("--no-hop-sweep", action="store_true")
    ap.add_argument("--hop-only", action="store_true", help="only the standalone hop table (wd_hop back to back), one JSON line")
    ap.add_argument("--no-config2", action="store_true", help="skip the configs[2] (12^4) force-evaluation time")
    return ap.parse_args()


def workload_name(cfg, n):
    lx, ly, lz, lt = cfg["dims"]
    return f"{lx}x{ly}x{lz}x{lt} SF lattice, eps={cfg['eps']}, kappa={cfg['kappa']}, n_rhs={n}, seed={cfg['seed']}"


# ------------------------------------------------------------------------------------------------
# the oracle, timed on the host cores (cpu_baseline leg and --impl reference arm)
# ------------------------------------------------------------------------------------------------
def pick_oracle_lattice(cfg, budget_s):
    """Largest L in (workload's L, 16, 12, 8) whose 1-RHS oracle force evaluation is expected to fit `budget_s` on this
    box: calibrated by timing the 8^4 case and scaling by (L/8)^4 x 1.6 (iteration counts and cache misses grow with L)."""
    t8, _ = oracle_force_eval(cfg, 8, 1)
    Lw = cfg["dims"][0]
    for L in sorted({Lw, 16, 12, 8}, reverse=True):
        if L <= Lw and (L == 8 or t8 * (L / 8.0) ** 4 * 1.6 <= budget_s):
            return L
    return 8


def oracle_force_eval(cfg, L, n_cols):
    """The oracle, as it stands, on `n_cols` right-hand sides of an L^4 SF lattice drawn from the workload's link / RHS
    distribution (its eps, kappa, seed; L = the workload's own lattice when it fits the time budget): both solves to
    TOL + force.  Returns (seconds, (iterations D, iterations D^dag) of column 0)."""
    import wd_inputs as wi
    from oracle import wd_oracle as orc
    dims = (L, L, L, L)
    U = wi.gauge_field(dims, cfg["eps"], cfg["seed"], cfg["bc"])
    Phi = wi.spinor_field(dims, n_cols, cfg["seed"], cfg["bc"])
    k, bc = cfg["kappa"], cfg["bc"]
    t0 = time.perf_counter()
    X, r1, it1, _ = orc.solve(dims, k, bc, 0, U, Phi, tol=TOL)
    Y, r2, it2, _ = orc.solve(dims, k, bc, 1, U, X, tol=TOL)
    orc.force(dims, k, bc, U, X, Y)
    return time.perf_counter() - t0, (int(it1[0]), int(it2[0]))


def oracle_apply_rate(cfg, n, threads=None):
    """site*RHS/s of the oracle's D apply on the workload's own lattice and n_rhs."""
    import wd_inputs as wi
    from oracle import wd_oracle as orc
    dims = cfg["dims"]
    U = wi.gauge_field(dims, cfg["eps"], cfg["seed"], cfg["bc"])
    Phi = wi.spinor_field(dims, n, cfg["seed"], cfg["bc"])
    full = orc.max_threads()
    if threads:
        orc.set_threads(threads)
    orc.apply(dims, cfg["kappa"], cfg["bc"], 0, U, Phi)
    t0 = time.perf_counter()
    reps = 2
    for _ in range(reps):
        orc.apply(dims, cfg["kappa"], cfg["bc"], 0, U, Phi)
    dt = (time.perf_counter() - t0) / reps
    orc.set_threads(full)
    lx, ly, lz, lt = dims
    return lx * ly * lz * lt * n / dt


def cpu_baseline(cfg, n, full=False):
    """cpu_baseline leg: ONE column of the workload's own lattice (the oracle solves column by column, so the block
    costs n_rhs times that: no extrapolation over lattice size), all host cores; plus the oracle's D-apply rate on the
    full block with all cores and with one thread, and a single-thread force evaluation on a stated smaller lattice."""
    from oracle import wd_oracle as orc
    Lw = cfg["dims"][0]
    cores = orc.max_threads()
    if full:
        L, ncol = Lw, n
    else:
        L, ncol = pick_oracle_lattice(cfg, 40.0), 1
    dt, iters = oracle_force_eval(cfg, L, ncol)
    orc.set_threads(1)
    Ls = 8 if Lw >= 8 else Lw
    dt1, it1 = oracle_force_eval(cfg, Ls, 1)
    orc.set_threads(cores)
    scale = (Lw / float(L)) ** 4 * n / ncol
    how = ("the whole workload" if full else
           f"1 of the {n} right-hand sides (the oracle works column by column, so the block costs {n} x that)" +
           ("" if L == Lw else f" on a {L}^4 lattice of the same distribution, scaled by site count x{(Lw / float(L)) ** 4:.2f} "
                               "(iteration counts grow slowly with L: this flatters the oracle)"))
    sample = (f"oracle (fp64, unpreconditioned BiCGStab, OpenMP over sites), {cores} threads: 2 solves to {TOL:g} + force on {how}: "
              f"{dt:.2f} s ({iters[0]}+{iters[1]} iterations for column 0)")
    return {"value": 1.0 / (dt * scale), "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
            "apply_site_rhs_per_s_all_cores": oracle_apply_rate(cfg, n),
            "apply_site_rhs_per_s_1_thread": oracle_apply_rate(cfg, n, threads=1),
            "single_thread": {"lattice": f"{Ls}^4 SF, 1 RHS", "seconds_per_force_eval": round(dt1, 2),
                              "iterations": list(it1)}}


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only).  Each step is a bounded sample: ONE right-hand side
    on the largest lattice of the workload's distribution that fits the time budget of this --steps/--warmup.  The line
    reports what was RUN (`value`, `ms_per_step`, `config.workload` are the sample's) and, separately, the estimate for
    the full workload (`scaled_to_full_workload`)."""
    from paper_1009_5169_b200 import replicas as rp
    if not rp.reference_arm_runs_here(rp.env_world()[1]):
        return
    import wd_inputs as wi
    from oracle import wd_oracle as orc
    cfg = dict(wi.CONFIGS[args.config])
    n = args.n_rhs
    L = pick_oracle_lattice(cfg, 150.0 / max(1, args.steps + args.warmup))
    for _ in range(args.warmup):
        oracle_force_eval(cfg, L, 1)
    times, iters = [], (0, 0)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        dt, iters = oracle_force_eval(cfg, L, 1)
        times.append(dt)
    total = time.perf_counter() - t0
    value = args.steps / sum(times)
    cores = orc.max_threads()
    lx, ly, lz, lt = cfg["dims"]
    scale = lx * ly * lz * lt * n / float(L ** 4)
    scfg = dict(cfg, dims=(L, L, L, L))
    sample = (f"each step = the oracle (fp64, unpreconditioned BiCGStab, OpenMP over sites) on 1 RHS of a {L}^4 SF lattice of the "
              f"workload's distribution: 2 solves to {TOL:g} + force, {sum(times) / len(times):.2f} s ({iters[0]}+{iters[1]} "
              f"iterations); value, ms_per_step and config.workload describe THIS sample")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 / value, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(scfg, 1), "full_workload": workload_name(cfg, n), "l2": "n/a (CPU)",
                   "sample_of_full_workload": f"1/{scale:.1f} of its site*RHS count"},
        "scaled_to_full_workload": {"value": value / scale, "unit": UNIT,
                                    "note": "by site*RHS count; iteration counts grow slowly with L, so this flatters the oracle"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": total,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        try:
            for ln in open(self.path):
                p = [x.strip() for x in ln.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1]))
                    smax.append(float(p[2]))
                except ValueError:
                    continue
                for name, v in zip(names, p[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(smax), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------------------------------------
# standalone hop (dslash) measurement: BASELINE.json metric "multi-RHS Wilson dslash GFLOP/s & HBM GB/s"
# ------------------------------------------------------------------------------------------------
def hop_bytes_per_launch(Vh, n, s, R, extra_operands=0.0, interior=1.0):
    """Algorithmic bytes of one hop launch on one output parity: per output site*RHS 24 reals in +
    24 out, +24 per extra operand the fused epilogue reads (xpay operand, left operand of a fused inner product), and
    8 links of R reals per site.  `interior` = (T-1)/T with Schroedinger-functional boundaries: the kernels skip the
    frozen t = 0 slice, so everything READ is counted on interior sites only; the output is written on all sites."""
    return Vh * (n * (24 * interior + 24 + 24 * extra_operands * interior) * s + 8 * R * s * interior)


def hop_sweep(pkg, ctx, torch, n, peak_gbs, reps=50, only=None, interior=1.0):
    """wd_hop back to back on native half-lattice blocks, fp32/fp64 x 18/12-real links; CUDA events
    on the launching stream.  Fields rotate through enough copies to exceed 2x L2 (L2-cold)."""
    res = {}
    Vh = ctx.V // 2
    precs = [(pkg.F32, "f32", 4), (pkg.F64, "f64", 8)]
    if ctx.native_numel(pkg.F32P, n) > 0:
        precs.insert(1, (pkg.F32P, "f32p", 4))   # two sites per thread, packed fp32 instructions (wd.h WD_F32P)
    for prec, pname, s in precs:
        if only and only[0] != pname:
            continue
        half = ctx.native_numel(prec, n) // 2
        dt = torch.float64 if prec == pkg.F64 else torch.float32
        nbuf = max(2, int(2 * 130e6 / (half * s)) + 1)
        bufs = [torch.randn(half, dtype=dt, device=ctx.device) for _ in range(nbuf)]
        out = [torch.empty(half, dtype=dt, device=ctx.device) for _ in range(2)]
        for recon, R in ((pkg.LINK18, 18), (pkg.LINK12, 12)):
            if only and only[1] != R:
                continue
            try:
                for i in range(5):
                    ctx.hop(pkg.OP_D, bufs[i % nbuf], n, 0, prec, recon, out=out[i % 2])
            except pkg.WdError:
                continue   # WD_F32P: the z-march kernel does not serve this shape
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for i in range(reps):
                ctx.hop(pkg.OP_D, bufs[i % nbuf], n, 0, prec, recon, out=out[i % 2])
            e1.record()
            torch.cuda.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / reps
            b = hop_bytes_per_launch(Vh, n, s, R, interior=interior)
            gbs = b / us * 1e-3
            res[f"{pname}_r{R}"] = {"us": round(us, 2), "gbs": round(gbs, 1), "frac_hbm": round(gbs / peak_gbs, 4),
                                    "gflops": round(1320.0 * Vh * n / us * 1e-3, 1),
                                    "site_rhs_per_s": round(Vh * n / us * 1e6, 0)}
        del bufs, out
    return res


def rhs_sweep(pkg, wi, torch, peak_gbs, R, recon):
    """BASELINE.json configs[4]: the blocked mixed-precision solve D X = Phi on 24^4 at n_rhs = 1, 2, 5, 8, 12:
    time per solve, per RHS and per inner iteration, and the standalone fp32 hop (L2-cold) at that n_rhs."""
    cfg = dict(wi.CONFIGS[4])
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    U = torch.from_numpy(wi.gauge_field(dims, cfg["eps"], cfg["seed"], bc)).cuda()
    out = {}
    for n in (1, 2, 5, 8, 12):
        ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n)
        ctx.set_gauge(U)
        P = ctx.pack(torch.from_numpy(wi.spinor_field(dims, n, cfg["seed"], bc)).cuda())
        X = torch.empty_like(P)
        for _ in range(2):
            ctx.solve_block(pkg.OP_D, P, n, tol=TOL, recon=recon, out=X)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        reps = 3
        for _ in range(reps):
            _, info = ctx.solve_block(pkg.OP_D, P, n, tol=TOL, recon=recon, out=X)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        del P, X
        hop = hop_sweep(pkg, ctx, torch, n, peak_gbs, reps=30, only=("f32", R), interior=(dims[3] - 1) / dims[3])
        out[str(n)] = {"solve_ms": round(ms, 3), "ms_per_rhs": round(ms / n, 3), "inner_iters": info["inner_iters_total"],
                       "us_per_inner_iter": round(ms * 1e3 / max(1, info["inner_iters_total"]), 1),
                       "max_relres": max(info["relres"]), "hop_f32": hop[f"f32_r{R}"]}
        ctx.close()
        del ctx
    return out


def apply_sweep(pkg, wi, torch, peak_gbs, reps=50):
    """BASELINE.json configs[3]: standalone D and D^dag apply (two hop launches, diagonal term fused) on the 16^4
    SF lattice, n_rhs = 5, fp32/fp64 x 18/12-real links.  L2-warm = same buffers every call (the 50-100 MB working
    set sits in the 126 MB L2); L2-cold = inputs rotated through more than 2x L2 of buffers.  GB/s counts the
    two-launch form: per site*RHS 72 reals (in twice, out once) plus 8 R reals of links per site."""
    cfg = dict(wi.CONFIGS[3])
    dims, kappa, bc, n = cfg["dims"], cfg["kappa"], cfg["bc"], 5
    U = torch.from_numpy(wi.gauge_field(dims, cfg["eps"], cfg["seed"], bc)).cuda()
    ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n)
    ctx.set_gauge(U)
    V = ctx.V
    res = {}
    for prec, pname, s in ((pkg.F32, "f32", 4), (pkg.F64, "f64", 8)):
        numel = ctx.native_numel(prec, n)
        dt = torch.float32 if prec == pkg.F32 else torch.float64
        nbuf = max(2, int(2 * 130e6 / (numel * s)) + 1)
        bufs = [torch.randn(numel, dtype=dt, device=ctx.device) for _ in range(nbuf)]
        out = torch.empty(numel, dtype=dt, device=ctx.device)
        for recon, R in ((pkg.LINK18, 18), (pkg.LINK12, 12)):
            for op, oname in ((pkg.OP_D, "D"), (pkg.OP_DDAG, "Ddag")):
                for mode in ("warm", "cold"):
                    for i in range(5):
                        ctx.apply(op, bufs[i % nbuf if mode == "cold" else 0], n, prec, recon, out=out)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize()
                    e0.record()
                    for i in range(reps):
                        ctx.apply(op, bufs[i % nbuf if mode == "cold" else 0], n, prec, recon, out=out)
                    e1.record()
                    torch.cuda.synchronize()
                    us = e0.elapsed_time(e1) * 1e3 / reps
                    b = V * (n * 72 * s + 8 * R * s)
                    res[f"{oname}_{pname}_r{R}_{mode}"] = {
                        "us": round(us, 2), "gbs": round(b / us * 1e-3, 1), "frac_hbm": round(b / us * 1e-3 / peak_gbs, 4),
                        "gflops": round(1368.0 * V * n / us * 1e-3, 1), "site_rhs_per_s": round(V * n / us * 1e6, 0)}
        del bufs, out
    ctx.close()
    return res


def config2_time(pkg, wi, torch, recon, idx=2):
    """BASELINE.json configs[idx] (2: the 12^4 SF lattice; 1: 8^4; 0: 4^4), 5 RHS: full MD force evaluation (two blocked
    solves + force).  L2-resident and launch-bound: an absolute time only, no roofline claim."""
    cfg, U, Phi = wi.make_config(idx)
    dims, kappa, bc, n = cfg["dims"], cfg["kappa"], cfg["bc"], cfg["n_rhs"]
    ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n)
    ctx.set_gauge(torch.from_numpy(U).cuda())
    P = ctx.pack(torch.from_numpy(Phi).cuda())
    for _ in range(2):
        X, Y, F, S, infos = ctx.md_force(P, n, recon=recon, want_action=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    reps = 5
    for _ in range(reps):
        X, Y, F, S, infos = ctx.md_force(P, n, recon=recon, want_action=False)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    ctx.close()
    return {"ms_per_force_eval": round(ms, 3), "inner_iters": [infos[0]["inner_iters_total"], infos[1]["inner_iters_total"]],
            "outer_steps": [infos[0]["outer_steps"], infos[1]["outer_steps"]],
            "max_relres": max(max(infos[0]["relres"]), max(infos[1]["relres"]))}


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_1009_5169_b200 as pkg
    import wd_inputs as wi

    from paper_1009_5169_b200 import replicas as rp
    world, rank, local = rp.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak_gbs = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"

    cfg = dict(wi.CONFIGS[args.config])
    cfg["seed"] = rp.replica_seed(cfg["seed"], rank)  # independent replica per rank
    n = args.n_rhs
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    recon = pkg.LINK12 if args.recon == 12 else pkg.LINK18
    R = args.recon
    U = wi.gauge_field(dims, cfg["eps"], cfg["seed"], bc)
    Phi = wi.spinor_field(dims, n, cfg["seed"], bc)

    ctx = pkg.Context(dims, kappa, bc=bc, max_rhs=n, device=f"cuda:{local}")
    if args.hop_impl >= 0:
        ctx.set_option(pkg.OPT_HOP_IMPL, args.hop_impl)
    ctx.set_gauge(torch.from_numpy(U).cuda())
    if args.hop_only:
        interior = (dims[3] - 1) / dims[3] if bc == wi.BC_SF else 1.0
        print(json.dumps({"hop": hop_sweep(pkg, ctx, torch, n, peak_gbs, interior=interior), "workload": workload_name(cfg, n),
                          "nvcc_defines": os.environ.get("WD_NVCC_DEFINES", ""), "peak_gbs": peak_gbs,
                          "note": "wd_hop back to back (50 launches per entry, L2-cold rotation), CUDA events"}))
        ctx.close()
        return
    Phi_host = torch.from_numpy(Phi).pin_memory()
    P = ctx.pack(Phi_host.cuda())
    X = torch.empty_like(P)
    Y = torch.empty_like(P)
    F = torch.zeros((4,) + tuple(reversed(dims)) + (3, 3, 2), dtype=torch.float64, device=ctx.device)
    F_host = torch.empty(F.shape, dtype=torch.float64).pin_memory()
    V = ctx.V
    Vh = V // 2

    def step():
        F.zero_()
        _, ix = ctx.solve_block(pkg.OP_D, P, n, tol=TOL, recon=recon, out=X)
        _, iy = ctx.solve_block(pkg.OP_DDAG, X, n, tol=TOL, recon=recon, out=Y)
        ctx.force(X, Y, n, F=F)
        return ix, iy

    def barrier():
        rp.barrier(dist, world)
        torch.cuda.synchronize()

    def max_over_ranks(ms):
        return rp.max_over_ranks(dist, torch, world, ms, ctx.device)

    for _ in range(max(args.warmup, 3)):
        ix, iy = step()
    # ---- timed region: device-resident inputs ---------------------------------------------------
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ix, iy = step()
    e1.record()
    barrier()
    launches = ctx.launch_count() - l0
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    ms_step = ms_total / args.steps
    value = rp.job_throughput(world, args.steps, ms_total)

    # ---- e2e: host buffers through the one-call C-ABI entry, copies inside the timed region --------
    # The links change between the force evaluations of a trajectory, so the end-to-end step uploads
    # and ingests the gauge field too (wd_md_force_host_gauge); the Phi-only form is reported beside it.
    U_host = torch.from_numpy(U).pin_memory()
    ctx.md_force_host_gauge(U_host, Phi_host, F_host, tol=TOL, recon=recon)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.md_force_host_gauge(U_host, Phi_host, F_host, tol=TOL, recon=recon)
    barrier()
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)
    e2e_value = rp.job_throughput(world, args.steps, e2e_ms)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.md_force_host(Phi_host, F_host, tol=TOL, recon=recon)
    barrier()
    e2e_phi_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)
    clocks = sampler.stop()
    f_check = float(F_host.abs().sum())
    assert np.isfinite(f_check) and f_check > 0.0
    # a0 alone: gauge upload (pinned host -> device) + ingest kernel
    Ud = torch.empty(U_host.shape, dtype=torch.float64, device=ctx.device)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(3):
        Ud.copy_(U_host, non_blocking=True)
        ctx.set_gauge(Ud)
    torch.cuda.synchronize()
    a0_ms = (time.perf_counter() - t0) * 1e3 / 3
    e0.record()
    for _ in range(3):
        ctx.set_gauge(Ud)
    e1.record()
    torch.cuda.synchronize()
    a0_ingest_ms = e0.elapsed_time(e1) / 3
    del Ud

    # ---- per-class device time of one more step (event pairs inside the library) -----------------
    ctx.profile(True)
    ix, iy = step()
    prof = ctx.profile_read()
    ctx.profile(False)
    hop_ms, hop_groups = prof["hop32"]
    # real fp32 hop launches of that step: 4 per BiCGStab iteration.  (The class also counts the no-op launches
    # enqueued between the last iteration and the next convergence poll; they must not dilute the average.)
    hop_cnt = 4 * (ix["inner_iters_total"] + iy["inner_iters_total"])
    tot_prof = sum(v[0] for v in prof.values())
    # the four fp32 hop launches of one BiCGStab iteration: plain, xpay + <rt, v> (2 extra operands), plain, and
    # xpay + <t, s>, <t, t> (1 extra operand: 0.75 per launch on average) or, in the merged-update schedule the solver
    # runs by default where the z-march kernel serves the hop, xpay + <t, s>, <t, t>, <rt, s>, <rt, t> (2 extra: 1.0)
    interior = (dims[3] - 1) / dims[3] if bc == wi.BC_SF else 1.0
    # schedule and kernel from the library's own dispatch (wd_inner_plan), not a copy of its rules: at 24^4 the z-march
    # kernel and the merged schedule serve n_rhs = 3, 5, 8, 10, while 4, 6, 12, 16 go to the ring kernel and the textbook order
    plan = ctx.inner_plan(n, recon)
    merged = plan["merged"]
    hop_bytes = hop_bytes_per_launch(Vh, n, 4, R, extra_operands=1.0 if merged else 0.75, interior=interior)
    hop_us = hop_ms * 1e3 / max(1, hop_cnt)
    achieved = hop_bytes / (hop_us * 1e-6) * 1e-9 if hop_cnt else 0.0
    kname = {"zmarch": f"hop_zm_kernel<float,{R}>", "ring": f"hop_tma_kernel<float,{R}>",
             "register": f"hop_kernel<float,{R}>"}[plan["hop_kernel"]]
    # dram__bytes_read.sum + dram__bytes_write.sum per launch from an ncu --set full capture of THIS kernel source: the
    # committed record carries the sha256 of the kernel's source file and is ignored when the source has changed since
    traffic, traffic_note, ncu_us = None, "no capture on record for this kernel source", None
    try:
        import hashlib
        tr = json.load(open(os.path.join(ROOT, "profiles", "r02_hop_traffic.json.txt")))
        src = {"hop_zm_kernel": "wd_hop_zm.cu", "hop_tma_kernel": "wd_hop_tma.cu", "hop_kernel": "wd_hop.cu"}[kname.split("<")[0]]
        sha = hashlib.sha256(open(os.path.join(ROOT, "paper_1009_5169_b200", "csrc", src), "rb").read()).hexdigest()
        if tr.get("kernel") == kname and tr.get("source_sha256") == sha and \
                tr.get("workload") == workload_name(dict(wi.CONFIGS[args.config]), n):
            traffic, traffic_note = tr["dram_bytes_per_launch"], tr.get("how", "")
            ncu_us = tr.get("ncu_us_per_launch")
        elif tr.get("source_sha256") != sha:
            traffic_note = "the capture on record is of an older kernel source"
    except Exception:
        pass
    roofline = {"bound": "hbm", "kernel": f"{kname} (fp32 multi-RHS Wilson hop inside the inner solver, 2 of 4 launches per iteration with "
                                          "fused xpay + inner-product epilogues)",
                "achieved": round(achieved, 1), "peak": peak_gbs, "unit": "GB/s", "frac": round(achieved / peak_gbs, 4),
                "peak_source": peak_src, "traffic": traffic, "traffic_note": traffic_note, "bytes_per_launch": hop_bytes,
                "bytes_counted": f"interior sites only for everything read ((T-1)/T = {interior:.4f}), all sites for the output",
                "avg_launch_us": round(hop_us, 2), "launches_in_step": hop_cnt,
                "schedule": "merged x,r,p update: 23 vector passes per iteration, 2 + 4 + 2 + 4 of them in the four hop launches" if merged
                            else "textbook order: 25 vector passes per iteration, 2 + 4 + 2 + 3 of them in the four hop launches",
                "timing": "CUDA event pairs on the library's stream around the two hop launches of every application of the "
                          "even/odd operator (one kernel-to-kernel gap inside each pair); in the graph-replayed blocks the pairs "
                          "are event-record nodes of the graph, read back after every replay",
                # the same four launches timed alone by ncu (gpu__time_duration of the committed full capture; cold caches,
                # no neighbours on the stream): context for how much of avg_launch_us is gap between dependent kernels
                "ncu_isolated": None if not ncu_us else {"avg_launch_us": round(sum(ncu_us) / len(ncu_us), 2),
                                                         "frac": round(hop_bytes / (sum(ncu_us) / len(ncu_us) * 1e-6) * 1e-9 / peak_gbs, 4)},
                "share_of_step": round(hop_ms / tot_prof, 4) if tot_prof else None,
                "gflops": round(1320.0 * Vh * n * interior / hop_us * 1e-3, 1) if hop_cnt else None}
    breakdown = {k: {"ms": round(v[0], 3), "launch_groups": v[1]} for k, v in prof.items()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(cfg, n), "inner_links": f"{R}-real fp32", "outer": "fp64 defect correction",
                   "launch": "inner iterations replayed as CUDA graphs, 4 per graph" if ctx.get_option(pkg.OPT_GRAPH) else "stream order",
                   "tol": TOL, "l2": "no flush: solver working set >> 126 MB L2", "parallelism": f"replicas x{world}"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms / args.steps,
                "h2d_bytes_per_step": (Phi_host.numel() + U_host.numel()) * 8, "d2h_bytes_per_step": F_host.numel() * 8,
                "includes": "gauge upload + ingest (a0), Phi upload + pack, both solves, force, F download",
                "phi_only_ms_per_step": e2e_phi_ms / args.steps},
        "a0_gauge": {"upload_plus_ingest_ms": round(a0_ms, 3), "ingest_kernel_ms": round(a0_ingest_ms, 3),
                     "h2d_bytes": U_host.numel() * 8},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "solver": {"outer_steps": [ix["outer_steps"], iy["outer_steps"]],
                   "inner_iters": [ix["inner_iters_total"], iy["inner_iters_total"]],
                   "max_relres": [max(ix["relres"]), max(iy["relres"])],
                   "site_rhs_per_s": V * n * value},
        "breakdown_ms": breakdown,
    }
    if rank == 0 and not args.no_hop_sweep:
        line["hop"] = hop_sweep(pkg, ctx, torch, n, peak_gbs, interior=interior)
    ctx.close()
    del ctx, P, X, Y, F
    sweeps = (world == 1 and not args.quick)
    if rank == 0 and (args.rhs_sweep or sweeps):
        line["rhs_sweep"] = rhs_sweep(pkg, wi, torch, peak_gbs, R, recon)
    if rank == 0 and (args.apply_sweep or sweeps):
        line["apply_16"] = apply_sweep(pkg, wi, torch, peak_gbs)
    if rank == 0 and not args.no_config2:
        line["config2_12x12x12x12"] = config2_time(pkg, wi, torch, recon)
        # the two smaller parity configurations beside it (launch-bound: what a persistent small-lattice mode would have to beat)
        line["config1_8x8x8x8"] = config2_time(pkg, wi, torch, recon, 1)
        line["config0_4x4x4x4"] = config2_time(pkg, wi, torch, recon, 0)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(dict(wi.CONFIGS[args.config]), n, full=args.cpu_baseline_full)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


def run_sharded(args):
    """--shard-rhs: the RHS-sharded multi-GPU form (paper_1009_5169_b200/sharded.py): one
    problem, its columns dealt to the ranks, one allReduce(sum) of F per force evaluation.  Total work is fixed: strong
    scaling.  The default N > 1 mode stays "replicas" (north_star: no sharding for the headline)."""
    import torch
    import torch.distributed as dist

    import paper_1009_5169_b200 as pkg
    import wd_inputs as wi
    from paper_1009_5169_b200 import replicas as rp
    from paper_1009_5169_b200 import sharded as sh
    world, rank, local = rp.env_world()
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = dict(wi.CONFIGS[args.config])
    n = args.n_rhs
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    recon = pkg.LINK12 if args.recon == 12 else pkg.LINK18
    dev = f"cuda:{local}"
    sc = sh.ShardedContext(pkg, dist, dims, kappa, bc, n, world, rank, dev)
    sc.set_gauge(torch.from_numpy(wi.gauge_field(dims, cfg["eps"], cfg["seed"], bc)).cuda())
    P = sc.pack_local(torch.from_numpy(wi.spinor_field(dims, n, cfg["seed"], bc)).cuda())
    for _ in range(max(args.warmup, 3)):
        F, S, infos = sc.md_force(P, recon=recon, tol=TOL)
    rp.barrier(dist, world)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        F, S, infos = sc.md_force(P, recon=recon, tol=TOL)
    e1.record()
    rp.barrier(dist, world)
    torch.cuda.synchronize()
    ms = rp.max_over_ranks(dist, torch, world, e0.elapsed_time(e1), sc.device)
    line = {"metric": METRIC, "value": args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_name(cfg, n), "parallelism": f"rhs-sharded x{world}: columns i mod {world}, gauge replicated, "
                       "allReduce(sum) of F", "columns_of_rank0": sh.columns_of_rank(n, world, 0), "tol": TOL},
            "exchange_bytes_per_step": 4 * 18 * 8 * dims[0] * dims[1] * dims[2] * dims[3], "action": S}
    sc.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.shard_rhs:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
