"""wcras_apply_D_noalloc (include/wcras.h, csrc/noalloc.cu): w = D v with the two internal-layout buffers in a file-scope
static device array instead of cudaMalloc'ed memory, for callers that may not allocate (CUDA graph capture, serving
loops).  Its output is compared with the existing path's (wcras_apply_D) on two calls in a row that share the array, and
the size limit is checked.  Named test_zz_* so that pytest collects it last; it builds its own contexts and passes alone
in a fresh process as well as after the other tests."""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu]

torch = pytest.importorskip("torch")

from paper_1011_3318_b200 import binding, inputs as I  # noqa: E402

TOL = {32: 2e-6, 64: 1e-13}   # the D-parity tolerances of tests/test_gpu_parity.py (TOL32, TOL64)


def make_ctx(which):
    cfg = I.CONFIGS[which]
    U = I.make_gauge(cfg)
    Ud = torch.view_as_real(torch.from_numpy(U)).contiguous().cuda()
    return cfg, binding.Context(cfg["dims"], cfg["kappa"], cfg["csw"], Ud)


def dev_spinor(dims, seed, prec):
    x = torch.view_as_real(torch.from_numpy(I.spinor(dims, seed)))
    return x.to(torch.float32 if prec == 32 else torch.float64).contiguous().cuda()


def rel(a, b):
    a, b = a.double().cpu().numpy(), b.double().cpu().numpy()
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("which", [0, 1])
@pytest.mark.parametrize("prec", [32, 64])
def test_apply_D_noalloc_matches_apply_D(which, prec):
    cfg, ctx = make_ctx(which)
    dims = cfg["dims"]
    x1, x2 = dev_spinor(dims, 101, prec), dev_spinor(dims, 102, prec)
    # new entry point FIRST (before wcras_apply_D has allocated anything for this context), two calls in a row: the second
    # starts from the array as the first left it
    y1, y2 = torch.full_like(x1, float("nan")), torch.full_like(x2, float("nan"))
    ctx.apply_D_noalloc(prec, x1, y1)
    ctx.apply_D_noalloc(prec, x2, y2)
    torch.cuda.synchronize()
    w1, w2 = torch.empty_like(x1), torch.empty_like(x2)
    ctx.apply_D(prec, x1, w1)
    ctx.apply_D(prec, x2, w2)
    torch.cuda.synchronize()
    for y, w in ((y1, w1), (y2, w2)):
        assert torch.isfinite(y).all()
        assert rel(y, w) <= TOL[prec]
        assert (y - w).abs().max().item() <= 10 * TOL[prec] * w.abs().max().item()
    assert rel(y1, w2) > 0.1   # the two calls really computed different things
    # and once more after the existing path has run, with the per-class timers on (the entry point switches them off)
    ctx.set_timing(True)
    y3 = torch.empty_like(x1)
    ctx.apply_D_noalloc(prec, x1, y3)
    ctx.set_timing(False)
    torch.cuda.synchronize()
    assert rel(y3, w1) <= TOL[prec]


def test_apply_D_noalloc_two_contexts_share_the_array():
    """Two contexts (different lattices, different precisions) alternate on the one array; calls are serialised on the
    stream, so each result is its own."""
    cfg0, c0 = make_ctx(0)
    cfg1, c1 = make_ctx(1)
    a, b = dev_spinor(cfg0["dims"], 103, 64), dev_spinor(cfg1["dims"], 104, 32)
    ya, yb, wa, wb = torch.empty_like(a), torch.empty_like(b), torch.empty_like(a), torch.empty_like(b)
    for _ in range(2):
        c1.apply_D_noalloc(32, b, yb)
        c0.apply_D_noalloc(64, a, ya)
    c0.apply_D(64, a, wa)
    c1.apply_D(32, b, wb)
    torch.cuda.synchronize()
    assert rel(ya, wa) <= TOL[64] and rel(yb, wb) <= TOL[32]


def test_apply_D_noalloc_size_limit_and_arguments():
    cfg, ctx = make_ctx(2)                    # 16^4 = 65536 sites: 12.6 MB at prec 32 (fits the 16 MiB array), 25.2 MB at 64
    dims = cfg["dims"]
    x32 = dev_spinor(dims, 105, 32)
    y32, w32 = torch.empty_like(x32), torch.empty_like(x32)
    ctx.apply_D_noalloc(32, x32, y32)
    ctx.apply_D(32, x32, w32)
    torch.cuda.synchronize()
    assert rel(y32, w32) <= TOL[32]
    x64 = dev_spinor(dims, 105, 64)
    y64 = torch.full_like(x64, 7.0)
    with pytest.raises(binding.WcrasError) as e:
        ctx.apply_D_noalloc(64, x64, y64)
    assert e.value.code == binding.UNSUPPORTED
    assert "static array" in str(e.value) and "16777216" in str(e.value)
    torch.cuda.synchronize()
    assert (y64 == 7.0).all()                 # nothing was launched
    for args in ((16, x32, y32), (32, x32, x32)):
        with pytest.raises(binding.WcrasError) as e:
            ctx.apply_D_noalloc(*args)
        assert e.value.code == binding.INVALID_ARG
