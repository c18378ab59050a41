"""BASELINE.json:configs[4] at full size (48^3 x 96, 10.6 M sites, ~60 GB of device memory; most of the run time is
the host-side generation of the synthetic gauge field and the oracle's field strength).

Always on (north_star: "true relative residual <= 1e-12 on every config"): D fp32/fp64 on sampled sites the oracle computes
one by one, the unpreconditioned solve and the RAS solve at the point configs[4] names (8^4 domains, overlap 1, 4 MR
iterations), each checked by the oracle's residual on the sampled sites beside the library's full-lattice fp64 residual.
WCRAS_BIG=1 adds the other preconditioner variants."""
import os

import numpy as np
import pytest

pytestmark = [pytest.mark.gpu]

torch = pytest.importorskip("torch")

import oracle as O  # noqa: E402
from paper_1011_3318_b200 import binding, inputs as I  # noqa: E402


def test_config4_full_size():
    cfg = I.CONFIGS[4]
    dims = cfg["dims"]
    V = I.volume(dims)
    U = I.make_gauge(cfg)
    Ud = torch.view_as_real(torch.from_numpy(U)).contiguous().cuda()
    ctx = binding.Context(dims, cfg["kappa"], cfg["csw"], Ud)
    del Ud
    torch.cuda.empty_cache()
    op = O.Operator(dims, U, cfg["kappa"], cfg["csw"])
    psi = I.spinor(dims, cfg["seed"])
    rng = np.random.default_rng(0)
    sites = np.array(sorted(set(int(s) for s in rng.integers(0, V, 400)) | {0, V - 1, dims[0] - 1, V - dims[0]}))
    want = op.apply_D_sites(psi, sites)

    def to_host(t):
        a = t.cpu().numpy()
        return (a[..., 0] + 1j * a[..., 1]).reshape(V, 4, 3)

    for prec, dt, tol in ((32, torch.float32, 2e-6), (64, torch.float64, 1e-13)):
        x = torch.view_as_real(torch.from_numpy(psi)).to(dt).contiguous().cuda()
        y = torch.empty_like(x)
        ctx.apply_D(prec, x, y)
        torch.cuda.synchronize()
        got = to_host(y)[sites].astype(np.complex128)
        assert np.linalg.norm(got - want) / np.linalg.norm(want) <= tol
        del x, y
    t32, t64 = ctx.time_kernel(0, 20), ctx.time_kernel(1, 10)
    print("\nD fp32 %.3f ms (%.0f GB/s)  fp64 %.3f ms (%.0f GB/s)" % (t32, 768 * V / t32 / 1e6, t64, 1536 * V / t64 / 1e6))

    eta_d = torch.view_as_real(torch.from_numpy(psi)).contiguous().cuda()
    phi_d = torch.empty_like(eta_d)

    def solve(label, warm=False):
        if warm:
            ctx.solve(eta_d, phi_d, 1e-12)
        i = ctx.solve(eta_d, phi_d, 1e-12)
        phi = to_host(phi_d)
        res = np.linalg.norm(psi[sites] - op.apply_D_sites(phi, sites)) / np.linalg.norm(psi[sites])
        print("%-40s %8.1f ms  inner %3d  K %3d  residual %.1e (oracle, sampled sites %.1e)" % (
            label, i["ms_total"], i["inner_iters"], i["ras_applies"], i["rel_resid_true"], res))
        assert i["status"] == 0 and i["rel_resid_true"] <= 1e-12 and res <= 3e-12
        return i

    big = os.environ.get("WCRAS_BIG") == "1"
    ctx.set_solver(use_ras=False)
    i0 = solve("no preconditioner", warm=big)
    ctx.set_solver(use_ras=True)
    r = cfg["ras"][0]                                     # the configuration BASELINE.json names: 8^4, overlap 1, 4 MR
    ctx.ras_precondition(r["domain"], r["overlap"], r["block_iters"], 1)
    i1 = solve("RAS 8^4 overlap 1 N_dominv 4 NRAS 1", warm=big)
    assert i1["inner_iters"] < i0["inner_iters"]          # the preconditioner cuts the Krylov iterations
    if not big:
        return
    ctx.ras_precondition((4, 4, 4, 4), 0, 2, 3)
    solve("RAS 4^4 overlap 0 N_dominv 2 NRAS 3", warm=True)
    ctx.set_operand_precision(16)
    ctx.ras_precondition((4, 4, 4, 4), 0, 2, 3)
    solve("RAS 4^4 overlap 0 N_dominv 2 NRAS 3, fp16 operands", warm=True)
    ctx.set_schwarz(True)
    ctx.ras_precondition((4, 4, 4, 4), 0, 3, 2)
    solve("SAP 4^4 N_dominv 3, 2 cycles, fp16 operands", warm=True)
    ctx.set_schwarz(False)
    ctx.ras_precondition(r["domain"], r["overlap"], r["block_iters"], 1)
    solve("RAS 8^4 overlap 1 N_dominv 4 NRAS 1, fp16 operands", warm=True)
    ctx.set_timing(True)   # per-class CUDA-event split of the same solve (profiles/r2_stream.md)
    i = solve("  the same with the class split on")
    ctx.set_timing(False)
    print("  class split: block solve %.1f ms (%d launches)  D fp32 %.1f  D fp64 %.1f  BLAS %.1f  of %.1f ms" % (
        i["ms_blocksolve"], i["ras_applies"], i["ms_dslash"], i["ms_dslash64"], i["ms_blas"], i["ms_total"]))
    ctx.set_operand_precision(32)
