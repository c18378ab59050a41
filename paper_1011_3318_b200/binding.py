"""Thin ctypes binding of libwcras (include/wcras.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libwcras.so.  There is no CPU fallback: if the shared
library is missing or no CUDA device is present, the calls raise.  PyTorch is used by the callers only to
own device memory and streams; the functions here accept anything with `data_ptr()` (torch tensors) or a
raw integer address.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# WCRAS_LIB: another build of the same library (e.g. the phase-profile build of `python -m paper_1011_3318_b200.build
# --phase-profile`); still a CUDA library behind the same C ABI, never a fallback
LIB_PATH = os.environ.get("WCRAS_LIB") or os.path.join(_HERE, "libwcras.so")

OK, INVALID_ARG, UNSUPPORTED, CUDA_ERROR, BREAKDOWN, NOT_CONVERGED = 0, -1, -2, -3, -4, -5

EXPORTS = [
    "wcras_create", "wcras_destroy", "wcras_apply_D", "wcras_apply_D_noalloc", "wcras_ras_precondition", "wcras_set_ras_tier", "wcras_set_operand_precision", "wcras_set_block_solver", "wcras_set_schwarz", "wcras_set_traversal",
    "wcras_apply_D_restricted", "wcras_ras_apply", "wcras_set_solver", "wcras_set_lookahead", "wcras_set_graphs", "wcras_set_timing", "wcras_solve",
    "wcras_solve_host", "wcras_solve_multi", "wcras_ras_autotune", "wcras_export_clover", "wcras_time_kernel", "wcras_launch_count", "wcras_last_error",
]


class WcrasInfo(C.Structure):
    _fields_ = [("outer_iters", C.c_int), ("inner_iters", C.c_int), ("inner_solves", C.c_int),
                ("dv_fp32", C.c_int), ("dv_fp64", C.c_int), ("block_dv", C.c_int), ("ras_applies", C.c_int),
                ("status", C.c_int), ("rel_resid_recur", C.c_double), ("rel_resid_true", C.c_double),
                ("ms_total", C.c_double), ("ms_dslash", C.c_double), ("ms_blocksolve", C.c_double),
                ("ms_blas", C.c_double), ("ms_dslash64", C.c_double)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class WcrasTuneRow(C.Structure):
    _fields_ = [("domain", C.c_int * 4), ("overlap_s", C.c_int), ("block_iters", C.c_int), ("nras", C.c_int),
                ("schwarz", C.c_int), ("operand_bits", C.c_int), ("block_solver", C.c_int), ("status", C.c_int), ("inner_iters", C.c_int), ("ras_applies", C.c_int), ("ms", C.c_double),
                ("rel_resid_true", C.c_double)]

    def asdict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_ if k != "domain"}
        d["domain"] = tuple(self.domain)
        return d


class WcrasError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libwcras error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """Load libwcras.so; raises if it has not been built (python -m paper_1011_3318_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libwcras.so is missing: build it with `python -m paper_1011_3318_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.wcras_last_error.restype = C.c_char_p
        lib.wcras_launch_count.restype = C.c_longlong
        _lib = lib
    return _lib


def _ptr(t):
    if t is None:
        return C.c_void_p(0)
    if isinstance(t, int):
        return C.c_void_p(t)
    return C.c_void_p(t.data_ptr())


def _i4(v):
    return (C.c_int * 4)(*[int(x) for x in v])


class Context:
    """One lattice + gauge field on one GPU (wcras_ctx)."""

    def __init__(self, dims, kappa, csw, gauge_dev, stream=None):
        self._lib = load()
        self._h = C.c_void_p(0)
        self.dims = tuple(int(d) for d in dims)
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        sp = C.c_void_p(0 if stream is None else int(getattr(stream, "cuda_stream", stream)))
        rc = self._lib.wcras_create(C.byref(self._h), _i4(dims), C.c_double(kappa), C.c_double(csw),
                                    _ptr(gauge_dev), sp)
        if rc:
            msg = self.last_error() if self._h else "wcras_create failed"
            if self._h:
                self._lib.wcras_destroy(self._h)
                self._h = C.c_void_p(0)
            raise WcrasError(rc, msg)

    def last_error(self) -> str:
        return self._lib.wcras_last_error(self._h).decode()

    def _chk(self, rc, allow=()):
        if rc and rc not in allow:
            raise WcrasError(rc, self.last_error())
        return rc

    def destroy(self):
        if self._h:
            self._lib.wcras_destroy(self._h)
            self._h = C.c_void_p(0)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def apply_D(self, prec, in_dev, out_dev):
        self._chk(self._lib.wcras_apply_D(self._h, C.c_int(prec), _ptr(in_dev), _ptr(out_dev)))

    def apply_D_noalloc(self, prec, in_dev, out_dev):
        self._chk(self._lib.wcras_apply_D_noalloc(self._h, C.c_int(prec), _ptr(in_dev), _ptr(out_dev)))

    def ras_precondition(self, domain, overlap, block_iters, nras=1):
        self._chk(self._lib.wcras_ras_precondition(self._h, _i4(domain), C.c_int(overlap), C.c_int(block_iters),
                                                   C.c_int(nras)))

    def set_block_solver(self, kind):
        self._chk(self._lib.wcras_set_block_solver(self._h, C.c_int(kind)))

    def set_ras_tier(self, tier):
        self._chk(self._lib.wcras_set_ras_tier(self._h, C.c_int(tier)))

    def set_operand_precision(self, bits):
        self._chk(self._lib.wcras_set_operand_precision(self._h, C.c_int(bits)))

    def set_traversal(self, ztile):
        self._chk(self._lib.wcras_set_traversal(self._h, C.c_int(ztile)))

    def set_schwarz(self, multiplicative):
        self._chk(self._lib.wcras_set_schwarz(self._h, C.c_int(1 if multiplicative else 0)))

    def apply_D_restricted(self, prec, domain_index, in_dev, out_dev):
        self._chk(self._lib.wcras_apply_D_restricted(self._h, C.c_int(prec), C.c_int(domain_index), _ptr(in_dev),
                                                     _ptr(out_dev)))

    def ras_apply(self, r_dev, v_dev):
        self._chk(self._lib.wcras_ras_apply(self._h, _ptr(r_dev), _ptr(v_dev)))

    def set_solver(self, inner_tol=5e-7, inner_maxit=1000, outer_maxit=50, use_ras=True):
        self._chk(self._lib.wcras_set_solver(self._h, C.c_double(inner_tol), C.c_int(inner_maxit),
                                             C.c_int(outer_maxit), C.c_int(1 if use_ras else 0)))

    def set_lookahead(self, iterations):
        self._chk(self._lib.wcras_set_lookahead(self._h, C.c_int(iterations)))

    def set_graphs(self, enable):
        self._chk(self._lib.wcras_set_graphs(self._h, C.c_int(1 if enable else 0)))

    def set_timing(self, enable):
        self._chk(self._lib.wcras_set_timing(self._h, C.c_int(1 if enable else 0)))

    def solve(self, eta_dev, phi_dev, tol, strict=True):
        info = WcrasInfo()
        rc = self._lib.wcras_solve(self._h, _ptr(eta_dev), _ptr(phi_dev), C.c_double(tol), C.byref(info))
        self._chk(rc, allow=() if strict else (NOT_CONVERGED, BREAKDOWN))
        return info.asdict()

    def solve_multi(self, nrhs, eta_dev, phi_dev, tol, strict=True):
        """nrhs stacked systems (wcras_solve_multi); returns (info, per-system true residuals)."""
        info = WcrasInfo()
        res = (C.c_double * nrhs)()
        rc = self._lib.wcras_solve_multi(self._h, C.c_int(nrhs), _ptr(eta_dev), _ptr(phi_dev), C.c_double(tol),
                                         C.byref(info), res)
        self._chk(rc, allow=() if strict else (NOT_CONVERGED, BREAKDOWN))
        return info.asdict(), list(res)

    def solve_host(self, eta_host_ptr, phi_host_ptr, tol, strict=True):
        """eta/phi: host buffers (numpy arrays via .ctypes.data, or pinned torch CPU tensors)."""
        info = WcrasInfo()
        rc = self._lib.wcras_solve_host(self._h, _ptr(eta_host_ptr), _ptr(phi_host_ptr), C.c_double(tol),
                                        C.byref(info))
        self._chk(rc, allow=() if strict else (NOT_CONVERGED, BREAKDOWN))
        return info.asdict()

    def ras_autotune(self, eta_dev, tol, max_rows=256):
        """Parameter survey (wcras_ras_autotune): returns (best row, list of all rows) and leaves best configured."""
        best = WcrasTuneRow()
        table = (WcrasTuneRow * max_rows)()
        n = C.c_int(0)
        self._chk(self._lib.wcras_ras_autotune(self._h, _ptr(eta_dev), C.c_double(tol), C.c_int(max_rows), C.byref(best),
                                               table, C.byref(n)))
        return best.asdict(), [table[k].asdict() for k in range(n.value)]

    def export_clover(self, out_dev):
        self._chk(self._lib.wcras_export_clover(self._h, _ptr(out_dev)))

    def time_kernel(self, which, reps) -> float:
        ms = C.c_double(0)
        self._chk(self._lib.wcras_time_kernel(self._h, C.c_int(which), C.c_int(reps), C.byref(ms)))
        return ms.value

    def launch_count(self) -> int:
        return int(self._lib.wcras_launch_count(self._h))
