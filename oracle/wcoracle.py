"""ctypes front end of oracle/wcoracle.c (argument marshalling only; all arithmetic is in the C file).

TEST INFRASTRUCTURE: see oracle/__init__.py.  Arrays are numpy complex128 in the canonical layouts
(gauge [V][4][3][3], spinor [V][4][3], field strength [V][6][3][3]); site index x fastest.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wcoracle.c")
_LIB = os.path.join(_HERE, "libwcoracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/wcoracle.c with gcc (-O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.wco_true_residual.restype = C.c_double
    return _lib


def _i4(v):
    return (C.c_int * 4)(*[int(t) for t in v])


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def volume(dims):
    return int(np.prod([int(d) for d in dims]))


def num_threads() -> int:
    return int(_load().wco_num_threads())


def gamma(mu: int) -> np.ndarray:
    """gamma_mu (mu=0..3) or gamma_5 (mu=4), 4x4."""
    out = np.zeros((4, 4), np.complex128)
    _load().wco_gamma(C.c_int(mu), _p(out))
    return out


def sigma(mu: int, nu: int) -> np.ndarray:
    out = np.zeros((4, 4), np.complex128)
    _load().wco_sigma(C.c_int(mu), C.c_int(nu), _p(out))
    return out


def round_half(a) -> np.ndarray:
    """Entrywise fp64 -> fp32 -> fp16 rounding (nearest even) of a complex array (wco_round_half)."""
    a = _c(a)
    out = np.empty_like(a)
    _load().wco_round_half(C.c_long(a.size), _p(a), _p(out))
    return out


def field_strength(dims, U) -> np.ndarray:
    U = _c(U)
    F = np.empty((volume(dims), 6, 3, 3), np.complex128)
    _load().wco_field_strength(_i4(dims), _p(U), _p(F))
    return F


class Operator:
    """Holds (dims, U, F, kappa, csw) for repeated calls."""

    def __init__(self, dims, U, kappa, csw):
        self.dims = tuple(int(d) for d in dims)
        self.V = volume(dims)
        self.U = _c(U).reshape(self.V, 4, 3, 3)
        self.kappa, self.csw = float(kappa), float(csw)
        self.F = field_strength(dims, self.U)

    def _args(self):
        return _i4(self.dims), _p(self.U), _p(self.F), C.c_double(self.kappa), C.c_double(self.csw)

    def clover_matrix(self) -> np.ndarray:
        """A(x) = 1 - (c_sw kappa/2) sum sigma (x) F as dense 12x12 matrices, [V][12][12] (wco_clover_matrix)."""
        A = np.empty((self.V, 12, 12), np.complex128)
        _load().wco_clover_matrix(_i4(self.dims), _p(self.F), C.c_double(self.kappa), C.c_double(self.csw), _p(A))
        return A

    def with_operands(self, U, A):
        """The same lattice and kappa with explicit links U [V][4][3][3] and site-diagonal matrices A [V][12][12]."""
        return ExplicitOperator(self, U, A)

    def rounded(self):
        """Reduced-precision operand variant (reading R1): links and A(x) rounded entrywise to fp16."""
        return self.with_operands(round_half(self.U), round_half(self.clover_matrix()))

    def apply_D(self, v):
        v = _c(v)
        out = np.empty((self.V, 4, 3), np.complex128)
        _load().wco_apply_D(*self._args(), _p(v), _p(out))
        return out

    def apply_D_sites(self, v, sites):
        v = _c(v)
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        out = np.empty((len(sites), 4, 3), np.complex128)
        _load().wco_apply_D_sites(*self._args(), _p(v), C.c_long(len(sites)), _p(sites), _p(out))
        return out

    def apply_D_box(self, start, ext, v):
        v = _c(v)
        out = np.empty((self.V, 4, 3), np.complex128)
        _load().wco_apply_D_box(*self._args(), _i4(start), _i4(ext), _p(v), _p(out))
        return out

    def domain_count(self, block):
        return int(_load().wco_domain_count(_i4(self.dims), _i4(block)))

    def domain_box(self, block, s, idx):
        o, st, ex = _i4([0] * 4), _i4([0] * 4), _i4([0] * 4)
        rc = _load().wco_domain_box(_i4(self.dims), _i4(block), C.c_int(s), C.c_int(idx), o, st, ex)
        if rc:
            raise ValueError("invalid domain decomposition")
        return tuple(o), tuple(st), tuple(ex)

    def apply_D_restricted(self, block, s, idx, v):
        """out = P'^T D_Omega'_idx P' v on full-lattice vectors."""
        _, st, ex = self.domain_box(block, s, idx)
        return self.apply_D_box(st, ex, v)

    def mr_block(self, start, ext, niter, r_full):
        """(v_local, rho_local) after niter MR iterations on the box; local index x fastest."""
        r_full = _c(r_full)
        n = int(np.prod(ext))
        v = np.empty((n, 4, 3), np.complex128)
        rho = np.empty((n, 4, 3), np.complex128)
        _load().wco_mr_block(*self._args(), _i4(start), _i4(ext), C.c_int(niter), _p(r_full), _p(v), _p(rho))
        return v, rho

    def mr2_block(self, start, ext, niter, r_full):
        """(v_local, rho_local) after niter D applications of the restarted two-dimensional minimal residual (GMRES(2),
        DESIGN.md reading R2) on the box; local index x fastest."""
        r_full = _c(r_full)
        n = int(np.prod(ext))
        v = np.empty((n, 4, 3), np.complex128)
        rho = np.empty((n, 4, 3), np.complex128)
        _load().wco_mr2_block(*self._args(), _i4(start), _i4(ext), C.c_int(niter), _p(r_full), _p(v), _p(rho))
        return v, rho

    def with_block_solver(self, kind):
        """The same operator with Alg. 1 / SAP / the solvers using block solver `kind`: "mr" or "mr2" (reading R2)."""
        import copy
        o = copy.copy(self)
        o._block_solver = {"mr": 0, "mr2": 1}[kind]
        return o

    def ras_apply(self, block, s, niter, nras, eta):
        eta = _c(eta)
        out = np.empty((self.V, 4, 3), np.complex128)
        rc = _load().wco_ras_apply(*self._args(), _i4(block), C.c_int(s), C.c_int(niter), C.c_int(nras),
                                   _p(eta), _p(out))
        if rc:
            raise ValueError("invalid domain decomposition")
        return out

    def sap_apply(self, block, niter, ncycle, eta):
        """Multiplicative Schwarz (SAP, PAPER.md:33 ref [5]), overlap 0, red-black domains."""
        eta = _c(eta)
        out = np.empty((self.V, 4, 3), np.complex128)
        rc = _load().wco_sap_apply(*self._args(), _i4(block), C.c_int(niter), C.c_int(ncycle), _p(eta), _p(out))
        if rc:
            raise ValueError("invalid or not two-colourable domain decomposition")
        return out

    def bicgstab(self, eta, tol=1e-12, maxit=10000, ras=None):
        """Flat fp64 BiCGStab; ras = None or dict(domain, overlap, block_iters, nras)."""
        eta = _c(eta)
        x = np.empty((self.V, 4, 3), np.complex128)
        counts = (C.c_long * 3)()
        resid = (C.c_double * 2)()
        r = ras or dict(domain=(0, 0, 0, 0), overlap=0, block_iters=0, nras=1)
        st = _load().wco_bicgstab(*self._args(), C.c_int(1 if ras else 0), _i4(r["domain"]), C.c_int(r["overlap"]),
                                  C.c_int(r["block_iters"]), C.c_int(r.get("nras", 1)), _p(eta), _p(x),
                                  C.c_double(tol), C.c_int(maxit), counts, resid)
        return x, dict(status=int(st), iters=counts[0], dv=counts[1], ras_applies=counts[2],
                       rel_resid_recur=resid[0], rel_resid_true=resid[1])

    def nested_bicgstab(self, eta, tol=1e-12, inner_tol=1e-5, inner_maxit=1000, outer_maxit=50, ras=None):
        eta = _c(eta)
        x = np.empty((self.V, 4, 3), np.complex128)
        counts = (C.c_long * 4)()
        resid = (C.c_double * 2)()
        r = ras or dict(domain=(0, 0, 0, 0), overlap=0, block_iters=0, nras=1)
        st = _load().wco_nested_bicgstab(*self._args(), C.c_int(1 if ras else 0), _i4(r["domain"]),
                                         C.c_int(r["overlap"]), C.c_int(r["block_iters"]), C.c_int(r.get("nras", 1)),
                                         _p(eta), _p(x), C.c_double(tol), C.c_double(inner_tol),
                                         C.c_int(inner_maxit), C.c_int(outer_maxit), counts, resid)
        return x, dict(status=int(st), outer_iters=counts[0], inner_iters=counts[1], dv=counts[2],
                       ras_applies=counts[3], rel_resid_recur=resid[0], rel_resid_true=resid[1])

    def true_residual(self, eta, phi) -> float:
        eta, phi = _c(eta), _c(phi)
        return float(_load().wco_true_residual(*self._args(), _p(eta), _p(phi)))


class ExplicitOperator(Operator):
    """Operator whose site-diagonal term is the stored matrix A(x) (wco_set_explicit_clover is set around every
    call into the C library and cleared afterwards); F and c_sw are not used."""

    def __init__(self, base, U, A):
        self.dims, self.V, self.kappa, self.csw = base.dims, base.V, base.kappa, base.csw
        self.U = _c(U).reshape(self.V, 4, 3, 3)
        self.F = base.F
        self.A = _c(A).reshape(self.V, 12, 12)

    def clover_matrix(self):
        return self.A.copy()


def _wrap_explicit(name):
    plain = getattr(Operator, name)

    def call(self, *a, **k):
        lib = _load()
        lib.wco_set_explicit_clover(_p(self.A))
        try:
            return plain(self, *a, **k)
        finally:
            lib.wco_set_explicit_clover(C.c_void_p(0))

    call.__name__ = name
    call.__doc__ = plain.__doc__
    return call


for _n in ("apply_D", "apply_D_sites", "apply_D_box", "mr_block", "mr2_block", "ras_apply", "sap_apply", "bicgstab",
           "nested_bicgstab", "true_residual"):
    setattr(ExplicitOperator, _n, _wrap_explicit(_n))


def _wrap_block_solver(cls, name):
    plain = getattr(cls, name)

    def call(self, *a, **k):
        kind = getattr(self, "_block_solver", 0)
        if not kind:
            return plain(self, *a, **k)
        lib = _load()
        lib.wco_set_block_solver(C.c_int(kind))
        try:
            return plain(self, *a, **k)
        finally:
            lib.wco_set_block_solver(C.c_int(0))

    call.__name__ = name
    call.__doc__ = plain.__doc__
    return call


for _cls in (Operator, ExplicitOperator):
    for _n in ("ras_apply", "sap_apply", "bicgstab", "nested_bicgstab"):
        setattr(_cls, _n, _wrap_block_solver(_cls, _n))
