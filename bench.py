#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

A "step" is one pass of the whole hot path: one mixed-precision nested BiCGStab solve of D phi = eta to true
residual <= 1e-12 on the 32^4 workload of BASELINE.json:configs[3] (kappa=0.1225, c_sw=1.0, Haar-random SU(3)
links seed 4, Gaussian source), RAS-preconditioned inner solver.  Inputs are synthetic (paper_1011_3318_b200/
inputs.py) and stand in for the paper's "random gauge configuration".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config4]

N > 1 (torchrun): replicas only -- every rank solves its own right-hand side on its own GPU, no data-path
collective (north_star: "no sharding and no inter-GPU collectives"); NCCL is used for the barrier and the
max-over-ranks timing.  --impl reference times the fp64 CPU oracle (oracle/): real 32^4 solves, as many of the
requested steps as fit a wall-clock budget (the line states how many were run).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "clover Dslash GB/s (% HBM peak); 32^4 RAS-BiCGStab time-to-1e-12"
TOL = 1e-12
# RAS parameters of the timed solve (every row states NRAS, Q10).  The timed step uses the fastest point of
# the paper's parameter survey (NRAS x N_dominv, here also over the domain shape and the operand
# storage) as found by wcras_ras_autotune on B200: it is NOT one of the two shapes configs[3] names; those are timed
# beside it (solve.named_shapes) and in the same interleaved loop as the unpreconditioned solve.
RAS = dict(domain=(4, 4, 4, 4), overlap=0, block_iters=2, nras=4)
OPERAND_BITS = 16   # block-solver operand storage of the timed step (reading R1); 32 is reported beside it
# the domain shapes configs[3] names, each at a few (N_dominv, NRAS) points of the paper's survey; the
# fastest point of every shape is what `ras_named_shapes_faster_than_no_prec` compares with the unpreconditioned solve
NAMED_SHAPES = [(8, 8, 4, 4), (8, 8, 8, 8)]
NAMED_POINTS = [(2, 3), (2, 4), (3, 2)]
SAP = dict(domain=(4, 4, 4, 4), block_iters=3, ncycle=2)
INNER_TOL = 5e-7
REFERENCE_BUDGET_S = 150.0   # wall-clock budget of the --impl reference arm
# dram__bytes_read.sum + dram__bytes_write.sum of one dslash_kernel<float> launch at 32^4 from the committed
# `ncu --set full` capture (profiles/r2_kernels.md); algorithmic bytes are 768 B/site = 805.3 MB
DSLASH_TRAFFIC_NCU_BYTES = 812.2e6
# dram__bytes_read.sum + dram__bytes_write.sum of ras_cta16_kernel, mean over the four launches of one K_RAS application
# (661 + 861 + 861 + 690 MB; profiles/r2_kernels.md): below the algorithmic 805 MB because L2 keeps part of the halo and rho_fin
BLOCK_TRAFFIC_NCU_BYTES = 768.3e6
KEYS = ("outer_iters", "inner_iters", "inner_solves", "dv_fp32", "dv_fp64", "block_dv", "ras_applies", "rel_resid_true",
        "ms_total")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", {}


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        self.p.wait()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def ras_label(r):
    return "%s_it%d_nras%d" % ("x".join(map(str, r["domain"])), r["block_iters"], r["nras"])


# ---------------------------------------------------------------------------------------------------------------
# the oracle as it stands, timed on the host cores (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------------
def oracle_solve_32(op, eta, n=1):
    """n real flat fp64 RAS-BiCGStab solves of the full 32^4 workload with the oracle (exact fp64 operands)."""
    ts, info = [], None
    for _ in range(n):
        t0 = time.time()
        _, info = op.bicgstab(eta, tol=TOL, ras=dict(RAS))
        ts.append(time.time() - t0)
    return ts, info


def cpu_sample_desc(cfg_id):
    return ("flat fp64 RAS-BiCGStab (domain %s, overlap %d, %d MR, NRAS %d) to 1e-12 on the FULL configs[%d] lattice, "
            "measured, not extrapolated" % ("x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"],
                                            RAS["nras"], cfg_id))


def run_reference(args, rank):
    if rank != 0:
        return
    import oracle as O
    from paper_1011_3318_b200 import inputs as I
    cfg = I.CONFIGS[3]
    dims = cfg["dims"]
    op = O.Operator(dims, I.make_gauge(cfg), cfg["kappa"], cfg["csw"])
    eta = I.spinor(dims, cfg["seed"])
    t_start = time.time()
    ts, info = oracle_solve_32(op, eta, 1)
    while len(ts) < args.steps and (time.time() - t_start) + ts[0] < REFERENCE_BUDGET_S:
        t2, info = oracle_solve_32(op, eta, 1)
        ts += t2
    ms = float(np.mean(ts)) * 1e3
    line = {
        "impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus, "steps": len(ts),
        "warmup": 0, "steps_requested": args.steps, "warmup_requested": args.warmup,
        "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3] 32^4 kappa=0.1225 c_sw=1.0 Haar SU(3) seed 4, RAS %s s=%d N_dominv=%d NRAS=%d, tol 1e-12"
                   % ("x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"], RAS["nras"]),
                   "note": "every step is one real oracle solve of the full lattice; %d of the %d requested steps fit the %.0f s "
                           "budget of this arm, no warm-up solves (a CPU loop nest has nothing to warm)" %
                           (len(ts), args.steps, REFERENCE_BUDGET_S)},
        "cpu_baseline": {"value": ms, "unit": "ms", "cores": O.num_threads(), "kind": "oracle", "sample": cpu_sample_desc(3),
                         "iters": int(info["iters"]), "dv": int(info["dv"]), "true_resid": float(info["rel_resid_true"]),
                         "seconds_each": ts},
        "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def oracle_table(torch, binding, I, O, config4=False):
    """SURVEY.md 8(d) / BASELINE.md 3: per config the oracle's apply_D (min of 5) and its flat fp64 BiCGStab with and
    without K_RAS, beside the GPU's D and nested solves at the RAS parameters BASELINE.json:configs names (NRAS 1)."""
    out = {}
    cores = O.num_threads()
    for cid in (0, 1, 2) + ((4,) if config4 else ()):
        cfg = I.CONFIGS[cid]
        dims = cfg["dims"]
        V = I.volume(dims)
        U = I.make_gauge(cfg)
        eta = I.spinor(dims, cfg["seed"])
        op = O.Operator(dims, U, cfg["kappa"], cfg["csw"])
        row = {"dims": "x".join(map(str, dims)), "sites": V}
        ts = []
        for _ in range(3 if cid == 4 else 5):
            t0 = time.time()
            op.apply_D(eta)
            ts.append(time.time() - t0)
        t = min(ts)
        row["oracle"] = {"cores": cores, "apply_D_ms": t * 1e3, "apply_D_gflops_1824": 1824.0 * V / t / 1e9,
                         "apply_D_gbs_1536": 1536.0 * V / t / 1e9}
        r = cfg["ras"][0]
        ras = dict(domain=r["domain"], overlap=r["overlap"], block_iters=r["block_iters"], nras=1)
        if cid != 4:
            for key, rr in (("no_prec", None), ("ras_" + ras_label(ras) + "_s%d" % ras["overlap"], ras)):
                t0 = time.time()
                _, i = op.bicgstab(eta, tol=TOL, ras=rr)
                row["oracle"][key] = {"seconds": time.time() - t0, "iters": int(i["iters"]), "dv": int(i["dv"]),
                                      "rel_resid_true": float(i["rel_resid_true"])}
        ctx = binding.Context(dims, cfg["kappa"], cfg["csw"], torch.view_as_real(torch.from_numpy(U)).contiguous().cuda())
        e = torch.view_as_real(torch.from_numpy(eta)).contiguous().cuda()
        p = torch.empty_like(e)
        g = {"dslash_fp32_us": ctx.time_kernel(0, 200) * 1e3, "dslash_fp64_us": ctx.time_kernel(1, 100) * 1e3}
        g["dslash_fp32_gbs_768"] = 768.0 * V / (g["dslash_fp32_us"] * 1e-6) / 1e9
        for key, rr in (("no_prec", None), ("ras_" + ras_label(ras) + "_s%d" % ras["overlap"], ras)):
            if rr is None:
                ctx.set_solver(inner_tol=INNER_TOL, use_ras=False)
            else:
                ctx.ras_precondition(rr["domain"], rr["overlap"], rr["block_iters"], rr["nras"])
                ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
            ctx.solve(e, p, TOL)
            ms = []
            for _ in range(5):
                i = ctx.solve(e, p, TOL)
                ms.append(i["ms_total"])
            g[key] = {k: i[k] for k in KEYS}
            g[key]["ms_total"] = float(np.median(ms))
            if cid != 4:
                a = p.cpu().numpy()
                g[key]["oracle_rel_resid_true"] = float(op.true_residual(eta, (a[..., 0] + 1j * a[..., 1]).reshape(V, 4, 3)))
        # every RAS point BASELINE.json:configs[cid] names (configs[1]: overlap 0 and 1; configs[2]: 4^4 vs 8x4x4x4, overlap
        # 0/1/2, block iterations 2-8), GPU solves with the oracle's residual of every solution; NRAS 1, fp32 operands
        if cid != 4:
            sweep = {}
            iters = (2, 4, 6, 8) if cid == 2 else (cfg["ras"][0]["block_iters"],)
            ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
            for rr in cfg["ras"]:
                for nit in iters:
                    ctx.ras_precondition(rr["domain"], rr["overlap"], nit, 1)
                    ctx.solve(e, p, TOL)
                    ms = []
                    for _ in range(3):
                        i = ctx.solve(e, p, TOL)
                        ms.append(i["ms_total"])
                    a = p.cpu().numpy()
                    sweep["ras_%s_s%d_it%d" % ("x".join(map(str, rr["domain"])), rr["overlap"], nit)] = {
                        "ms_total": float(np.median(ms)), "inner_iters": i["inner_iters"], "ras_applies": i["ras_applies"],
                        "rel_resid_true": i["rel_resid_true"],
                        "oracle_rel_resid_true": float(op.true_residual(eta, (a[..., 0] + 1j * a[..., 1]).reshape(V, 4, 3)))}
            g["named_points"] = sweep
        row["gpu"] = g
        out["config%d" % cid] = row
        del ctx, e, p
    return out


def run_survey(torch, binding, I):
    """The paper's parameter survey as the library runs it (wcras_ras_autotune): every row tried on the BASELINE field
    (configs[3]) and on the near-critical field of `hard_regime`, with fp16 and fp32 operand storage as the starting point."""
    cfg = I.CONFIGS[3]
    dims = cfg["dims"]
    out = {"survey": "wcras_ras_autotune, tol 1e-12, 32^4", "fields": {}}
    for name, U, kappa, csw, seed in (("configs[3] (Haar links, kappa 0.1225)", I.make_gauge(cfg), cfg["kappa"], cfg["csw"], cfg["seed"]),
                                      ("near-critical (links exp(i 0.2 H) seed 17, kappa 0.13)", I.gauge_exp(dims, 0.2, 17), 0.13, 1.0, 18)):
        ctx = binding.Context(dims, kappa, csw, torch.view_as_real(torch.from_numpy(U)).contiguous().cuda())
        eta = torch.view_as_real(torch.from_numpy(I.spinor(dims, seed))).contiguous().cuda()
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
        ctx.set_operand_precision(16)
        t0 = time.time()
        best, rows = ctx.ras_autotune(eta, TOL, max_rows=256)
        out["fields"][name] = {"seconds": time.time() - t0, "best": best, "rows": rows}
        del ctx, eta
        torch.cuda.empty_cache()
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg and the oracle table")
    ap.add_argument("--no-hard", action="store_true", help="skip the near-critical side rows (a second gauge field)")
    ap.add_argument("--no-side", action="store_true", help="skip the side rows (named shapes, SAP, multi-RHS, configs 0-2)")
    ap.add_argument("--config4", action="store_true", help="add configs[4] (48^3 x 96, minutes of host time) to `configs`")
    ap.add_argument("--survey", action="store_true",
                    help="run the parameter survey (wcras_ras_autotune, PAPER.md:109) on configs[3] and on the near-critical field "
                         "and print its rows as one JSON line instead of the benchmark (profiles/r2_survey.md)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    from paper_1011_3318_b200 import binding, inputs as I, replicas as R

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if args.survey:
        run_survey(torch, binding, I)
        return
    if world > 1:
        R.init("nccl", torch.device("cuda", local))
    hbm_peak, peak_src, peaks_json = peaks()

    cfg = I.CONFIGS[3]
    dims = cfg["dims"]
    V = I.volume(dims)
    U = I.make_gauge(cfg)
    eta = I.spinor(dims, cfg["seed"], stream=R.source_streams(rank, world)[0])  # independent right-hand side per replica
    stream = torch.cuda.current_stream()
    Ud = torch.view_as_real(torch.from_numpy(U)).contiguous().cuda()
    ctx = binding.Context(dims, cfg["kappa"], cfg["csw"], Ud, stream=stream)
    del Ud
    eta_d = torch.view_as_real(torch.from_numpy(eta)).contiguous().cuda()
    phi_d = torch.empty_like(eta_d)
    eta_h = torch.view_as_real(torch.from_numpy(eta)).contiguous().pin_memory()
    phi_h = torch.empty_like(eta_h).pin_memory()
    warm = max(args.warmup, 3)

    def barrier():
        R.barrier(world, cuda=True)

    def max_over_ranks(x):
        return R.max_over_ranks(x, world, "cuda")

    def configure(r, bits, sap=False):
        ctx.set_operand_precision(bits)
        ctx.set_schwarz(sap)
        ctx.ras_precondition(r["domain"], r.get("overlap", 0), r["block_iters"], r["nras"] if "nras" in r else r["ncycle"])
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)

    def measure(n=3):
        """one warm-up solve, then n solves: the last info with the median / min / max of ms_total"""
        ctx.solve(eta_d, phi_d, TOL)
        ms, i = [], None
        for _ in range(n):
            i = ctx.solve(eta_d, phi_d, TOL)
            ms.append(i["ms_total"])
        d = {k: i[k] for k in KEYS}
        d.update(ms_total=float(np.median(ms)), ms_min=float(min(ms)), ms_max=float(max(ms)), solves=n)
        return d

    ctx.set_timing(False)
    side = {}
    if not args.no_side:
        # ---- the domain shapes configs[3] names (cluster tier), multiplicative Schwarz, stacked right-hand sides ----
        for dom in NAMED_SHAPES:
            best = None
            for (nit, nras) in NAMED_POINTS:     # fp16 operand storage: cluster tier with TMA staging (ras_cl16.cu)
                rp = dict(domain=dom, overlap=0, block_iters=nit, nras=nras)
                configure(rp, 16)
                m = measure()
                side["ras_%s_op16" % ras_label(rp)] = m
                if best is None or m["ms_total"] < best[1]:
                    best = (rp, m["ms_total"])
            configure(best[0], 32)               # the same point with fp32 operands (ras_fused.cu)
            side["ras_%s_op32" % ras_label(best[0])] = measure()
        for bits in (32, 16):
            configure(SAP, bits, sap=True)
            side["sap_%s_it%d_ncycle%d_op%d" % ("x".join(map(str, SAP["domain"])), SAP["block_iters"], SAP["ncycle"], bits)] = measure()
        # the second block solver (wcras_set_block_solver(1), reading R2: restarted two-dimensional minimal
        # residual) at the SAP point above and at the timed RAS point: same iteration counts on this well-conditioned field,
        # so it only costs its three extra dots here; it pays on the near-critical field (hard_regime)
        ctx.set_block_solver(1)
        configure(SAP, 16, sap=True)
        side["sap_%s_it%d_ncycle%d_op16_mr2" % ("x".join(map(str, SAP["domain"])), SAP["block_iters"], SAP["ncycle"])] = measure()
        configure(RAS, 16)
        side["ras_%s_op16_mr2" % ras_label(RAS)] = measure()
        ctx.set_block_solver(0)
        ctx.set_schwarz(False)
        configure(RAS, 32)
        side["ras_%s_op32" % ras_label(RAS)] = measure()
        if world == 1:
            etas4 = np.stack([I.spinor(dims, cfg["seed"], stream=k) for k in range(4)])
            e4 = torch.view_as_real(torch.from_numpy(etas4)).contiguous().cuda()
            p4 = torch.empty_like(e4)
            for bits in (32, 16):   # 32: stacked kernels (operands loaded once per 4 spinors); 16: the staged fp16 kernel per right-hand side
                configure(RAS, bits)
                ctx.solve_multi(4, e4, p4, TOL)
                i4, res4 = ctx.solve_multi(4, e4, p4, TOL)
                side["ras_multi_rhs_4_op%d" % bits] = {"ms_total": i4["ms_total"], "ms_per_rhs": i4["ms_total"] / 4,
                                                        "inner_iters": i4["inner_iters"], "ras_applies": i4["ras_applies"],
                                                        "worst_rel_resid_true": max(res4)}
            del e4, p4, etas4

    # ---- the timed step: RAS-preconditioned nested solve, per-class event timing OFF ----
    configure(RAS, OPERAND_BITS)
    for _ in range(warm):
        ctx.solve(eta_d, phi_d, TOL)
    barrier()
    l0 = ctx.launch_count()
    sampler = ClockSampler(torch.cuda.current_device()) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    infos = []
    e0.record(stream)
    for _ in range(args.steps):
        infos.append(ctx.solve(eta_d, phi_d, TOL))
    e1.record(stream)
    barrier()
    ms_step = max_over_ranks(e0.elapsed_time(e1) / args.steps)
    launches = (ctx.launch_count() - l0)
    clocks = sampler.stop() if sampler else None
    info = infos[-1]

    # ---- the same solve and the unpreconditioned one, interleaved, same flags, same number of solves ----
    pair = {"ras": [], "no_prec": []}
    info_np = None
    for _ in range(args.steps):
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
        pair["ras"].append(ctx.solve(eta_d, phi_d, TOL)["ms_total"])
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=False)
        info_np = ctx.solve(eta_d, phi_d, TOL)
        pair["no_prec"].append(info_np["ms_total"])
    ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)

    def stats(x):
        return {"mean": float(np.mean(x)), "median": float(np.median(x)), "min": float(min(x)), "max": float(max(x)), "n": len(x)}

    # ---- end to end: host buffers, H2D of eta and D2H of phi inside the timed region ----
    ctx.solve_host(eta_h, phi_h, TOL)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        ctx.solve_host(eta_h, phi_h, TOL)
    e1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1) / args.steps)

    # ---- per-kernel-class split (separate pass with the event timers ON) and burst timings ----
    ctx.set_timing(True)
    split = [ctx.solve(eta_d, phi_d, TOL) for _ in range(3)]
    ctx.set_timing(False)
    n_dv = sum(i["dv_fp32"] for i in split)
    ms_dslash_in_solve = sum(i["ms_dslash"] for i in split) / max(1, n_dv)
    n_blk = sum(i["block_dv"] for i in split) // RAS["block_iters"]
    ms_blk_in_solve = sum(i["ms_blocksolve"] for i in split) / max(1, n_blk)
    # a whole K_RAS application back to back, as the inner solver issues it (the class split above puts an event record
    # between the launches, which undoes the programmatic dependent launch of the chained cycles).  Measured right behind
    # the solves and for as many applications as one solve has (7), median of 5: behind a few hundred back-to-back launches
    # of the burst timings below the board is power-capped and the same launches take 10 % longer than inside a solve
    ms_kras = float(np.median([ctx.time_kernel(4, 7) for _ in range(5)]))
    ms_blk_chained = ms_kras / RAS["nras"]
    ms_d32 = ctx.time_kernel(0, 100)
    ms_d64 = ctx.time_kernel(1, 50)
    ms_blk = ctx.time_kernel(2, 50)
    ms_blas = ctx.time_kernel(3, 100)
    gbs_in_solve = 768.0 * V / (ms_dslash_in_solve * 1e-3) / 1e9
    gbs_burst = 768.0 * V / (ms_d32 * 1e-3) / 1e9
    true_resid = info["rel_resid_true"]
    # algorithmic HBM bytes per site of one block-solver launch: operands + residual in + v out,
    # chained cycles add rho_fin, the halo slots (96 B per site each way at 4^4: every face site) and the phi read-modify-write
    ob = 288 if OPERAND_BITS == 16 else 576
    nmid = max(0, RAS["nras"] - 2)
    cyc_bytes = [ob + 96 + 96 + 96 + 96] + [ob + 96 + 96 + 96 + 96 + 192] * nmid + [ob + 96 + 96 + 192]   # cycle 0, middle, last
    blk_bytes_in_solve = float(np.mean(cyc_bytes))
    blk_bytes_plain = ob + 96 + 96
    # the same launches against the FP32 pipe: 648 packed-pair instructions (FFMA2 / FADD2 / FMUL2, two
    # lane-cycles each) per site and MR sweep, 108 more per site for the boundary coupling of a chained cycle (60 in, 48 out)
    sm_hz = 1e6 * float((clocks or {}).get("sm_mhz") or peaks_json.get("sm_max_mhz") or 1965.0)
    alu_peak = 148 * 128 * sm_hz                                      # FP32 lane-cycles per second
    alu_cycles = [2.0 * (648 * RAS["block_iters"] + c) for c in [48] + [108] * nmid + [60]]   # cycle 0 (halo out), middle, last (halo in)
    alu_cycles_in_solve = float(np.mean(alu_cycles))

    if rank != 0:
        R.shutdown(world)
        return

    # ---- the paper's regime beside it: a smooth, near-critical field (hundreds of iterations, like Table 1) ----
    hard = None
    if world == 1 and not args.no_hard:
        del ctx
        torch.cuda.empty_cache()
        Uh = I.gauge_exp(dims, 0.2, 17)
        ch = binding.Context(dims, 0.13, 1.0, torch.view_as_real(torch.from_numpy(Uh)).contiguous().cuda(), stream=stream)
        eh = torch.view_as_real(torch.from_numpy(I.spinor(dims, 18))).contiguous().cuda()
        ph = torch.empty_like(eh)
        hard = {"workload": "32^4, links exp(i 0.2 H) seed 17, kappa=0.13 c_sw=1, Gaussian source seed 18, tol 1e-12"}

        def hrun(key):
            ch.solve(eh, ph, TOL)
            i = ch.solve(eh, ph, TOL)
            hard[key] = {k: i[k] for k in ("inner_iters", "ras_applies", "dv_fp32", "rel_resid_true", "ms_total")}

        ch.set_solver(inner_tol=INNER_TOL, use_ras=False)
        hrun("no_prec")
        ch.set_solver(inner_tol=INNER_TOL, use_ras=True)
        for bits in (32, 16):
            ch.set_operand_precision(bits)
            ch.ras_precondition((4, 4, 4, 4), 0, 5, 3)     # the paper's best point: NRAS 3, N_dominv 5
            hrun("ras_4x4x4x4_it5_nras3_op%d" % bits)
        for dom in ((8, 8, 4, 4), (8, 8, 8, 8)):        # the domain shapes configs[3] names (cluster tier)
            for bits in (32, 16):
                ch.set_operand_precision(bits)
                ch.ras_precondition(dom, 0, 5, 3)
                hrun("ras_%s_it5_nras3_op%d" % ("x".join(map(str, dom)), bits))
        ch.set_operand_precision(16)
        ch.ras_precondition((4, 4, 4, 4), 0, 5, 3)
        ch.set_schwarz(True)
        hrun("sap_4x4x4x4_it5_ncycle3_op16")
        ch.set_block_solver(1)                       # second block solver (reading R2) at its best surveyed points here
        ch.ras_precondition((4, 4, 4, 4), 0, 6, 3)
        hrun("sap_4x4x4x4_it6_ncycle3_op16_mr2")
        ch.set_schwarz(False)
        ch.ras_precondition((4, 4, 4, 4), 0, 4, 3)
        hrun("ras_4x4x4x4_it4_nras3_op16_mr2")
        ch.set_block_solver(0)
        del ch, eh, ph
        torch.cuda.empty_cache()

    cpu, configs = None, None
    if world == 1 and not args.no_cpu:
        import oracle as O
        if not args.no_side:
            configs = oracle_table(torch, binding, I, O, args.config4)
        op = O.Operator(dims, U, cfg["kappa"], cfg["csw"])
        ts = []
        for _ in range(5):
            t0 = time.time()
            op.apply_D(eta)
            ts.append(time.time() - t0)
        tD = min(ts)
        t_solve, oi = oracle_solve_32(op, eta, 1)
        t0 = time.time()
        _, oi_np = op.bicgstab(eta, tol=TOL, ras=None)
        t_np = time.time() - t0
        cpu = {"value": t_solve[0] * 1e3, "unit": "ms", "cores": O.num_threads(), "kind": "oracle", "sample": cpu_sample_desc(3),
               "iters": int(oi["iters"]), "dv": int(oi["dv"]), "true_resid": float(oi["rel_resid_true"]),
               "no_prec": {"value": t_np * 1e3, "unit": "ms", "iters": int(oi_np["iters"]), "dv": int(oi_np["dv"])},
               "apply_D_ms": tD * 1e3, "apply_D_gflops_1824": 1824.0 * V / tD / 1e9, "apply_D_gbs_1536": 1536.0 * V / tD / 1e9}

    np_med = float(np.median(pair["no_prec"]))
    named_faster = {}
    for dom in NAMED_SHAPES:
        pre = "ras_%s_" % "x".join(map(str, dom))
        rows = {k: v["ms_total"] for k, v in side.items() if k.startswith(pre)}
        if rows:
            kb = min(rows, key=rows.get)
            named_faster["x".join(map(str, dom))] = {"best": kb, "ms": rows[kb], "no_prec_ms": np_med, "faster": rows[kb] < np_med}
    line = {
        "metric": METRIC, "value": ms_step, "unit": "ms", "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 inner / f64 outer", "data": "synthetic",
        "config": {"workload": "configs[%d]: %s lattice, kappa=%g c_sw=%g, Haar SU(3) links seed %d, Gaussian source; RAS "
                               "domain %s overlap %d N_dominv %d NRAS %d, block-solver operands stored as fp%d; inner_tol %g; "
                               "tol 1e-12; replicas only (one RHS per GPU)"
                               % (3, "x".join(map(str, dims)), cfg["kappa"], cfg["csw"], cfg["seed"],
                                  "x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"], RAS["nras"], OPERAND_BITS,
                                  INNER_TOL),
                   "ras_point": "fastest point of the parameter survey (wcras_ras_autotune, PAPER.md:109); NOT a shape configs[3] "
                                "names -- the named shapes 8x8x4x4 and 8^4 are in solve.named_shapes",
                   "l2": "inputs larger than L2 (links+clover 604 MB fp32 per Dslash pass, 302 MB fp16 per block-solver launch)"},
        "clocks": clocks,
        "e2e": {"value": ms_e2e, "unit": "ms", "h2d_bytes_per_step": int(eta_h.numel() * 8),
                "d2h_bytes_per_step": int(phi_h.numel() * 8)},
        "gpu_launches": int(launches),
        # fp32 clover Dslash: 768 B/site; inside the solve every launch also carries a fused dot (it reads a
        # fourth vector: 864 B/site, frac_fused_variant) and its time includes the dot_finish_kernel behind it
        "roofline": {"kernel": "dslash_kernel<float> (fp32 clover Dslash)", "bound": "hbm", "achieved": gbs_in_solve,
                     "peak": hbm_peak, "peak_source": peak_src, "unit": "GB/s", "frac": gbs_in_solve / hbm_peak,
                     "traffic": DSLASH_TRAFFIC_NCU_BYTES, "algorithmic_bytes": 768.0 * V,
                     "bytes_per_site": 768, "sites": V,
                     "ms_per_launch_in_solve": ms_dslash_in_solve, "ms_per_launch_burst": ms_d32,
                     "frac_fused_variant": 864.0 * V / (ms_dslash_in_solve * 1e-3) / 1e9 / hbm_peak,
                     "achieved_burst": gbs_burst, "frac_burst": gbs_burst / hbm_peak,
                     "frac_of_nominal_8TBs": gbs_burst / 8000.0,
                     "gflops_1824_per_site": 1824.0 * V / (ms_d32 * 1e-3) / 1e9},
        # the kernel the timed solve spends most of its time in: one K_RAS cycle over all domains
        "roofline_block_solve": {
            "kernel": "ras_cta16_kernel (persistent one-CTA-per-domain MR block solver, fp%d operands staged by TMA, %d sweeps "
                      "per launch)" % (OPERAND_BITS, RAS["block_iters"]),
            "bound": "hbm", "unit": "GB/s", "sites": V, "peak": hbm_peak,
            "bytes_per_site_in_solve": blk_bytes_in_solve, "bytes_per_site_by_cycle": cyc_bytes,
            "traffic": BLOCK_TRAFFIC_NCU_BYTES, "algorithmic_bytes": blk_bytes_in_solve * V,
            "ms_per_launch_in_solve": ms_blk_chained, "ms_per_k_ras_application": ms_kras,
            "ms_per_launch_class_split": ms_blk_in_solve,
            "achieved": blk_bytes_in_solve * V / (ms_blk_chained * 1e-3) / 1e9,
            "frac": blk_bytes_in_solve * V / (ms_blk_chained * 1e-3) / 1e9 / hbm_peak,
            "frac_fp32_equivalent_864": 864.0 * V / (ms_blk_chained * 1e-3) / 1e9 / hbm_peak,
            "bytes_per_site_plain": blk_bytes_plain, "ms_per_launch_burst": ms_blk,
            "frac_burst": blk_bytes_plain * V / (ms_blk * 1e-3) / 1e9 / hbm_peak,
            "site_sweeps_per_s_burst": V * RAS["block_iters"] / (ms_blk * 1e-3),
            "alu": {"bound": "alu", "unit": "FP32 lane-cycles/s", "peak": alu_peak, "peak_source": "148 SMs x 128 FP32 lanes x SM clock",
                    "lane_cycles_per_site_by_cycle": alu_cycles, "achieved": alu_cycles_in_solve * V / (ms_blk_chained * 1e-3),
                    "frac": alu_cycles_in_solve * V / (ms_blk_chained * 1e-3) / alu_peak,
                    "frac_burst": 2.0 * 648 * RAS["block_iters"] * V / (ms_blk * 1e-3) / alu_peak,
                    "hbm_floor_ms": blk_bytes_in_solve * V / hbm_peak / 1e6, "alu_floor_ms": alu_cycles_in_solve * V / alu_peak * 1e3},
            "note": "ms_per_launch_in_solve = median of 5 timings of 7 K_RAS applications (one solve's worth, CUDA events on the "
                    "library's stream) right behind the timed solves, / NRAS; ms_per_launch_class_split = the same launches inside "
                    "the solves of the class-split pass (an event record between launches); ms_per_launch_burst = 50 plain "
                    "launches back to back behind the Dslash burst timings (board power-capped by then); "
                    "frac = algorithmic bytes actually moved by the fp16-operand kernel; frac_fp32_equivalent_864 prices the same "
                    "launch at the 864 B/site of the fp32-operand kernel it replaces (VERDICT r1 item 1); the HBM floor is the "
                    "larger of the two floors (alu.hbm_floor_ms against alu.alu_floor_ms), so the bound is 'hbm'; what the kernel "
                    "is limited by in practice is latency at 2 warps per scheduler (255 registers x 256 threads), see profiles/"},
        "cpu_baseline": cpu,
        "solve": {"ras": {k: info[k] for k in KEYS},
                  "class_split_ms": {"note": "separate pass with wcras_set_timing(1), mean of 3 solves",
                                     "dslash": float(np.mean([i["ms_dslash"] for i in split])),
                                     "dslash64": float(np.mean([i["ms_dslash64"] for i in split])),
                                     "blocksolve": float(np.mean([i["ms_blocksolve"] for i in split])),
                                     "blas": float(np.mean([i["ms_blas"] for i in split])),
                                     "total": float(np.mean([i["ms_total"] for i in split]))},
                  "no_prec": {k: info_np[k] for k in KEYS if k in info_np},
                  "interleaved_ms": {"ras": stats(pair["ras"]), "no_prec": stats(pair["no_prec"])},
                  "ras_faster_than_no_prec": float(np.median(pair["ras"])) < float(np.median(pair["no_prec"])),
                  "ras_named_shapes_faster_than_no_prec": named_faster,
                  "named_shapes": side},
        # vector passes (96 B per site each) of one inner BiCGStab iteration in its right-preconditioned form (p^, s^ stored):
        # SURVEY.md 8(d) budgets 10-12 for the fused form against ~19 unfused
        "blas_vector_passes_per_inner_iteration": {"k_update_p": 4, "k_update_s": 3, "k_update_xr": 8, "dot_operands_read_by_the_two_dslash": 2,
                                                   "total": 17, "unfused_same_recurrence": 24,
                                                   "note": "r,p,v->p; r,v->s (+|s|^2); x,p^,s^,s,t,rt->x,r (+<rt,r>,|r|^2); <rt,v> and <t,s>,<t,t> "
                                                           "ride on the Dslash that produces v and t; the first iteration skips k_update_p (p = b)"},
        "kernels": {"dslash_fp32_ms": ms_d32, "dslash_fp64_ms": ms_d64,
                    "dslash_fp64_gbs": 1536.0 * V / (ms_d64 * 1e-3) / 1e9,
                    "block_solve_ms": ms_blk,
                    "blas_update_xr_ms": ms_blas, "blas_update_xr_gbs": 8 * 96.0 * V / (ms_blas * 1e-3) / 1e9},
        "configs": configs,
        "hard_regime": hard,
        "true_residual": true_resid,
    }
    print(json.dumps(line))
    R.shutdown(world)


if __name__ == "__main__":
    main()
