#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

A "step" is one pass of the whole hot path: one mixed-precision nested BiCGStab solve of D phi = eta to true
residual <= 1e-12 on the 32^4 workload of BASELINE.json:configs[3] (kappa=0.1225, c_sw=1.0, Haar-random SU(3)
links seed 4, Gaussian source), RAS-preconditioned inner solver.  Inputs are synthetic (paper_1011_3318_b200/
inputs.py) and stand in for the paper's "random gauge configuration".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

N > 1 (torchrun): replicas only -- every rank solves its own right-hand side on its own GPU, no data-path
collective (north_star: "no sharding and no inter-GPU collectives"); NCCL is used for the barrier and the
max-over-ranks timing.  --impl reference times the fp64 CPU oracle (oracle/) on a bounded sample.
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
# RAS parameters of the timed solve (every row states NRAS, Q10)
# The timed step uses the fastest point of the paper's parameter survey (NRAS x N_dominv, here also
# over the domain shape) as measured on B200; the domain shapes BASELINE.json:configs[3] names are timed beside it.
RAS = dict(domain=(4, 4, 4, 4), overlap=0, block_iters=2, nras=3)
RAS_NAMED = [dict(domain=(8, 8, 4, 4), overlap=0, block_iters=3, nras=2),
             dict(domain=(8, 8, 8, 8), overlap=0, block_iters=5, nras=1)]
SAP = dict(domain=(4, 4, 4, 4), block_iters=3, ncycle=2)
INNER_TOL = 5e-7
# dram__bytes_read.sum + dram__bytes_write.sum of one dslash_kernel<float> launch at 32^4 from the committed
# `ncu --set full` capture (profiles/r1j_kernels.md); algorithmic bytes are 768 B/site = 805.3 MB
DSLASH_TRAFFIC_NCU_BYTES = 810.3e6


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


def cpu_sample(cfg_id, steps=1):
    """The oracle as it stands, on a bounded sample: the 16^4 sub-volume of the same workload (same kappa, c_sw,
    gauge recipe/seed, source recipe, RAS parameters), flat fp64 RAS-BiCGStab to 1e-12.  Returns seconds per
    solve at 16^4 and the x16 per-site extrapolation to 32^4 (iteration counts are nearly volume independent on
    these random fields; stated in `sample`)."""
    import oracle as O
    from paper_1011_3318_b200 import inputs as I
    cfg = I.CONFIGS[cfg_id]
    dims = tuple(min(16, d) for d in cfg["dims"])
    scale = I.volume(cfg["dims"]) / I.volume(dims)
    U = I.make_gauge(cfg, dims)
    eta = I.spinor(dims, cfg["seed"])
    op = O.Operator(dims, U, cfg["kappa"], cfg["csw"])
    ts, info = [], None
    for _ in range(steps):
        t0 = time.time()
        _, info = op.bicgstab(eta, tol=TOL, ras=dict(RAS))
        ts.append(time.time() - t0)
    t = float(np.mean(ts))
    return dict(seconds_sample=t, seconds_scaled=t * scale, cores=O.num_threads(), iters=int(info["iters"]),
                dv=int(info["dv"]), true_resid=float(info["rel_resid_true"]),
                sample="flat fp64 RAS-BiCGStab (domain %s, overlap %d, %d MR, NRAS %d) to 1e-12 on the %s sub-volume of "
                       "the workload (1/%d of the sites), time scaled x%d per site" %
                       ("x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"], RAS["nras"],
                        "x".join(map(str, dims)), int(scale), int(scale)))


def run_reference(args, rank):
    if rank != 0:
        return
    ts = []
    c = None
    for k in range(args.warmup + args.steps):
        c = cpu_sample(args.config, 1)
        if k >= args.warmup:
            ts.append(c["seconds_scaled"] * 1e3)
    ms = float(np.mean(ts))
    line = {
        "impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[%d] 32^4 kappa=0.1225 c_sw=1.0 Haar SU(3) seed 4, RAS %s s=%d N_dominv=%d NRAS=%d, tol 1e-12"
                   % (args.config, "x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"], RAS["nras"])},
        "cpu_baseline": {"value": ms, "unit": "ms", "cores": c["cores"], "kind": "oracle", "sample": c["sample"],
                         "iters": c["iters"], "dv": c["dv"]},
        "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-hard", action="store_true", help="skip the near-critical side rows (a second gauge field)")
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
    if world > 1:
        R.init("nccl", torch.device("cuda", local))
    hbm_peak, peak_src, peaks_json = peaks()

    cfg = I.CONFIGS[args.config]
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

    def barrier():
        R.barrier(world, cuda=True)

    def max_over_ranks(x):
        return R.max_over_ranks(x, world, "cuda")

    # ---- unpreconditioned solve, for the side-by-side row (not the timed step) ----
    ctx.set_solver(inner_tol=INNER_TOL, use_ras=False)
    ctx.set_timing(False)
    ctx.solve(eta_d, phi_d, TOL)
    info_noprec = ctx.solve(eta_d, phi_d, TOL)

    # ---- the domain shapes configs[3] names, for the side-by-side rows (not the timed step) ----
    named = {}
    for rp in RAS_NAMED:
        ctx.ras_precondition(rp["domain"], rp["overlap"], rp["block_iters"], rp["nras"])
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
        ctx.solve(eta_d, phi_d, TOL)
        i = ctx.solve(eta_d, phi_d, TOL)
        named["ras_%s_it%d_nras%d" % ("x".join(map(str, rp["domain"])), rp["block_iters"], rp["nras"])] = {
            k: i[k] for k in ("outer_iters", "inner_iters", "inner_solves", "dv_fp32", "dv_fp64", "block_dv", "ras_applies",
                              "rel_resid_true", "ms_total")}

    # ---- multiplicative Schwarz (SAP) beside it: same kernel, red-black half steps ----
    ctx.set_schwarz(True)
    ctx.ras_precondition(SAP["domain"], 0, SAP["block_iters"], SAP["ncycle"])
    ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
    ctx.solve(eta_d, phi_d, TOL)
    i = ctx.solve(eta_d, phi_d, TOL)
    named["sap_%s_it%d_ncycle%d" % ("x".join(map(str, SAP["domain"])), SAP["block_iters"], SAP["ncycle"])] = {
        k: i[k] for k in ("outer_iters", "inner_iters", "inner_solves", "dv_fp32", "dv_fp64", "block_dv", "ras_applies",
                          "rel_resid_true", "ms_total")}
    ctx.set_schwarz(False)

    # ---- four right-hand sides as one stacked solve, RAS point of the timed step ----
    if world == 1:
        etas4 = np.stack([I.spinor(dims, cfg["seed"], stream=k) for k in range(4)])
        e4 = torch.view_as_real(torch.from_numpy(etas4)).contiguous().cuda()
        p4 = torch.empty_like(e4)
        ctx.ras_precondition(RAS["domain"], RAS["overlap"], RAS["block_iters"], RAS["nras"])
        ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
        ctx.solve_multi(4, e4, p4, TOL)
        i4, res4 = ctx.solve_multi(4, e4, p4, TOL)
        named["ras_multi_rhs_4"] = {"ms_total": i4["ms_total"], "ms_per_rhs": i4["ms_total"] / 4, "inner_iters": i4["inner_iters"],
                                    "ras_applies": i4["ras_applies"], "worst_rel_resid_true": max(res4)}
        del e4, p4

    # ---- the timed step: RAS-preconditioned nested solve ----
    ctx.ras_precondition(RAS["domain"], RAS["overlap"], RAS["block_iters"], RAS["nras"])
    ctx.set_solver(inner_tol=INNER_TOL, use_ras=True)
    ctx.set_timing(True)
    for _ in range(max(args.warmup, 3)):
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

    # ---- end to end: host buffers, H2D of eta and D2H of phi inside the timed region ----
    ctx.set_timing(False)
    ctx.solve_host(eta_h, phi_h, TOL)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        ctx.solve_host(eta_h, phi_h, TOL)
    e1.record(stream)
    barrier()
    ms_e2e = max_over_ranks(e0.elapsed_time(e1) / args.steps)

    # ---- per-kernel numbers ----
    n_dv = sum(i["dv_fp32"] for i in infos)
    ms_dslash_in_solve = sum(i["ms_dslash"] for i in infos) / max(1, n_dv)
    ms_d32 = ctx.time_kernel(0, 100)
    ms_d64 = ctx.time_kernel(1, 50)
    ms_blk = ctx.time_kernel(2, 50)
    ms_blas = ctx.time_kernel(3, 100)
    n_blk = sum(i["block_dv"] for i in infos) // RAS["block_iters"]
    ms_blk_in_solve = sum(i["ms_blocksolve"] for i in infos) / max(1, n_blk)
    # inside the solve every fp32 D launch is the variant with the fused dot (<rt,v> or <t,s>,<t,t>): it also reads
    # the dot vector, 864 B/site, and its time includes the one-CTA dot_finish_kernel launched behind it
    gbs_in_solve = 864.0 * V / (ms_dslash_in_solve * 1e-3) / 1e9
    gbs_burst = 768.0 * V / (ms_d32 * 1e-3) / 1e9
    true_resid = info["rel_resid_true"]

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
        ch.ras_precondition((4, 4, 4, 4), 0, 5, 3)     # the paper's best point: NRAS 3, N_dominv 5
        hrun("ras_4x4x4x4_it5_nras3")
        for dom in ((8, 8, 4, 4), (8, 8, 8, 8)):        # the domain shapes configs[3] names (cluster tier)
            ch.ras_precondition(dom, 0, 5, 3)
            hrun("ras_%s_it5_nras3" % "x".join(map(str, dom)))
        ch.ras_precondition((4, 4, 4, 4), 0, 5, 3)
        ch.set_schwarz(True)
        hrun("sap_4x4x4x4_it5_ncycle3")
        del ch, eh, ph

    cpu = None
    if world == 1 and not args.no_cpu:
        c = cpu_sample(args.config, 1)
        cpu = {"value": c["seconds_scaled"] * 1e3, "unit": "ms", "cores": c["cores"], "kind": "oracle",
               "sample": c["sample"], "iters": c["iters"], "dv": c["dv"], "sample_seconds": c["seconds_sample"]}

    line = {
        "metric": METRIC, "value": ms_step, "unit": "ms", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32 inner / f64 outer", "data": "synthetic",
        "config": {"workload": "configs[%d]: %s lattice, kappa=%g c_sw=%g, Haar SU(3) links seed %d, Gaussian source; RAS "
                               "domain %s overlap %d N_dominv %d NRAS %d; inner_tol %g; tol 1e-12; replicas only (one RHS per GPU)"
                               % (args.config, "x".join(map(str, dims)), cfg["kappa"], cfg["csw"], cfg["seed"],
                                  "x".join(map(str, RAS["domain"])), RAS["overlap"], RAS["block_iters"], RAS["nras"], INNER_TOL),
                   "l2": "inputs larger than L2 (links+clover 604 MB fp32 per Dslash pass)"},
        "clocks": clocks,
        "e2e": {"value": ms_e2e, "unit": "ms", "h2d_bytes_per_step": int(eta_h.numel() * 8),
                "d2h_bytes_per_step": int(phi_h.numel() * 8)},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "dslash_kernel<float> (fp32 clover Dslash)", "bound": "hbm", "achieved": gbs_in_solve,
                     "peak": hbm_peak, "peak_source": peak_src, "unit": "GB/s", "frac": gbs_in_solve / hbm_peak,
                     "traffic": DSLASH_TRAFFIC_NCU_BYTES if V == 1 << 20 else None, "algorithmic_bytes": 768.0 * V,
                     "bytes_per_site": 768, "bytes_per_site_in_solve": 864, "sites": V,
                     "ms_per_launch_in_solve": ms_dslash_in_solve, "ms_per_launch_burst": ms_d32,
                     "achieved_burst": gbs_burst, "frac_burst": gbs_burst / hbm_peak,
                     "frac_of_nominal_8TBs": gbs_burst / 8000.0,
                     "gflops_1824_per_site": 1824.0 * V / (ms_d32 * 1e-3) / 1e9},
        # the kernel the timed solve spends most of its time in (profiles/): one K_RAS cycle over all domains
        "roofline_block_solve": {
            "kernel": "ras_cta_kernel (persistent one-CTA-per-domain MR block solver, %d sweeps per launch)" % RAS["block_iters"],
            "bound": "hbm", "unit": "GB/s", "bytes_per_site": 864, "sites": V, "peak": hbm_peak,
            "ms_per_launch_in_solve": ms_blk_in_solve, "achieved": 864.0 * V / (ms_blk_in_solve * 1e-3) / 1e9,
            "frac": 864.0 * V / (ms_blk_in_solve * 1e-3) / 1e9 / hbm_peak,
            "ms_per_launch_burst": ms_blk, "frac_burst": 864.0 * V / (ms_blk * 1e-3) / 1e9 / hbm_peak,
            "note": "HBM floor = operands 576 + r 96 + v 96 + phi/rho 96 B per site; the kernel is bound by fp32 issue "
                    "latency at 2 warps per scheduler, see profiles/r1j_kernels.md"},
        "cpu_baseline": cpu,
        "solve": {"ras": {k: info[k] for k in ("outer_iters", "inner_iters", "inner_solves", "dv_fp32", "dv_fp64", "block_dv",
                                              "ras_applies", "rel_resid_true", "ms_total", "ms_dslash", "ms_dslash64",
                                              "ms_blocksolve", "ms_blas")},
                  "no_prec": {k: info_noprec[k] for k in ("outer_iters", "inner_iters", "inner_solves", "dv_fp32", "dv_fp64",
                                                          "rel_resid_true", "ms_total")},
                  "ras_faster_than_no_prec": info["ms_total"] < info_noprec["ms_total"], **named},
        "kernels": {"dslash_fp32_ms": ms_d32, "dslash_fp64_ms": ms_d64,
                    "dslash_fp64_gbs": 1536.0 * V / (ms_d64 * 1e-3) / 1e9,
                    "block_solve_ms": ms_blk,
                    "block_solve_site_sweeps_per_s": V * RAS["block_iters"] / (ms_blk * 1e-3),
                    "block_solve_hbm_gbs": 864.0 * V / (ms_blk * 1e-3) / 1e9,
                    "blas_update_xr_ms": ms_blas, "blas_update_xr_gbs": 8 * 96.0 * V / (ms_blas * 1e-3) / 1e9},
        "hard_regime": hard,
        "true_residual": true_resid,
    }
    print(json.dumps(line))
    R.shutdown(world)


if __name__ == "__main__":
    main()
