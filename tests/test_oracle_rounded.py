"""Pins for the reduced-precision operand variant of the oracle (reading R1):
wco_round_half (fp64 -> fp32 -> fp16, nearest even), wco_clover_matrix (A(x) written out as a dense matrix) and the
explicit-A code path (wco_set_explicit_clover).  CPU only.  Checked against things the oracle does not compute in
that code: numpy's IEEE binary16, hand-worked ties, the test's own Kronecker construction of A(x), and the
already pinned formula path of the oracle.
"""
import numpy as np

import oracle as O
from paper_1011_3318_b200 import inputs as I
from test_oracle_operator import TG


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def test_round_half_hand_worked_cases():
    """Ties to even, gradual underflow, largest finite value: worked by hand from the binary16 format
    (11-bit significand, spacing 2^-10 in [1,2), smallest subnormal 2^-24, largest finite 65504)."""
    cases = [
        (1.0, 1.0), (-1.0, -1.0), (0.0, 0.0),
        (1 + 2.0 ** -11, 1.0),                      # tie between 1 and 1 + 2^-10: even significand
        (1 + 3 * 2.0 ** -11, 1 + 2 * 2.0 ** -10),   # tie between 1 + 2^-10 and 1 + 2^-9: even significand
        (1 + 2.0 ** -11 + 2.0 ** -20, 1 + 2.0 ** -10),   # just above the tie
        (2.0 ** -25, 0.0), (3 * 2.0 ** -25, 2.0 ** -23), (2.0 ** -24, 2.0 ** -24),   # subnormals
        (2.0 ** -14 * (1 + 2.0 ** -11), 2.0 ** -14),      # smallest normal binade, tie to even
        (65504.0, 65504.0), (0.1, 0.0999755859375), (-0.3, -0.300048828125),
        # double rounding (reading Q16: fp32 first): 1 + 2^-11 + 2^-30 rounds to 1 + 2^-11 in fp32, a tie -> 1,
        # whereas direct fp64 -> fp16 rounding would give 1 + 2^-10
        (1 + 2.0 ** -11 + 2.0 ** -30, 1.0),
    ]
    x = np.array([c[0] for c in cases]) + 0j
    want = np.array([c[1] for c in cases])
    got = O.round_half(x)
    assert np.array_equal(got.real, want) and np.all(got.imag == 0)
    z = O.round_half(np.array([0.1 - 0.3j]))
    assert z[0] == 0.0999755859375 - 0.300048828125j          # real and imaginary parts separately


def test_round_half_matches_numpy_binary16():
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.standard_normal(20000), rng.standard_normal(20000) * 1e-3, rng.standard_normal(5000) * 1e-6,
                        1 + rng.standard_normal(20000) * 1e-2, rng.uniform(-2, 2, 20000),
                        (rng.integers(-4096, 4096, 5000) + 0.5) * 2.0 ** -11])    # exact ties in [-2, 2]
    want = x.astype(np.float32).astype(np.float16).astype(np.float64)
    got = O.round_half(x + 1j * x[::-1])
    assert np.array_equal(got.real, want) and np.array_equal(got.imag, want[::-1])
    assert np.array_equal(O.round_half(got), got)                # idempotent


def test_clover_matrix_is_the_kronecker_formula():
    """A(x) = 1 - (c_sw kappa/2) sum_{mu<nu} sigma_mu_nu (x) F_mu_nu(x), built here with the test's own gamma matrices."""
    dims = (4, 4, 2, 6)
    kappa, csw = 0.121, 1.3
    op = O.Operator(dims, I.gauge_exp(dims, 0.6, 41), kappa, csw)
    A = op.clover_matrix()
    planes = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    want = np.zeros((op.V, 12, 12), complex) + np.eye(12)
    for p, (m, n) in enumerate(planes):
        sig = 0.5j * (TG[m] @ TG[n] - TG[n] @ TG[m])
        want -= (csw * kappa / 2) * np.einsum("ab,vij->vaibj", sig, op.F[:, p]).reshape(op.V, 12, 12)
    assert np.abs(A - want).max() < 1e-15
    assert np.abs(A - A.conj().transpose(0, 2, 1)).max() < 1e-15           # Hermitian
    assert np.abs(A[:, :6, 6:]).max() == 0 and np.abs(A[:, 6:, :6]).max() == 0   # two chiral blocks
    assert np.abs(A - np.eye(12)).max() > 1e-3                             # not trivially the identity


def test_explicit_path_reproduces_formula_path():
    """With unrounded operands the explicit-A code path is the pinned formula path: D, D_Omega', MR, Alg. 1, SAP,
    BiCGStab, residual.  (A transposed or conjugated A, or a mix-up of sites, fails here: A is Hermitian, not symmetric.)"""
    dims = (4, 4, 4, 6)
    op = O.Operator(dims, I.gauge_exp(dims, 0.6, 42), 0.12, 1.1)
    ex = op.with_operands(op.U, op.clover_matrix())
    psi = I.spinor(dims, 43)
    assert rel(ex.apply_D(psi), op.apply_D(psi)) < 1e-15
    sites = np.array([0, 5, 77, op.V - 1])
    assert rel(ex.apply_D_sites(psi, sites), op.apply_D_sites(psi, sites)) < 1e-15
    assert rel(ex.apply_D_restricted((2, 2, 2, 3), 1, 3, psi), op.apply_D_restricted((2, 2, 2, 3), 1, 3, psi)) < 1e-15
    assert rel(ex.ras_apply((2, 2, 2, 3), 1, 3, 2, psi), op.ras_apply((2, 2, 2, 3), 1, 3, 2, psi)) < 1e-13
    assert rel(ex.sap_apply((2, 2, 2, 3), 3, 2, psi), op.sap_apply((2, 2, 2, 3), 3, 2, psi)) < 1e-13
    x0, i0 = op.bicgstab(psi, tol=1e-12, ras=dict(domain=(2, 2, 2, 3), overlap=0, block_iters=2, nras=2))
    x1, i1 = ex.bicgstab(psi, tol=1e-12, ras=dict(domain=(2, 2, 2, 3), overlap=0, block_iters=2, nras=2))
    assert i0["iters"] == i1["iters"] and rel(x1, x0) < 1e-10
    assert abs(ex.true_residual(psi, x0) - op.true_residual(psi, x0)) < 1e-15
    # the global switch is cleared after every call: the formula path is unaffected afterwards
    assert rel(op.apply_D(psi), ex.apply_D(psi)) < 1e-15


def test_rounded_operator():
    """The rounded operator is the exact operator of the rounded fields: a perturbation of relative size ~2^-11, still
    gamma5-Hermitian (entrywise rounding commutes with conjugation), and equal to D built from the rounded links when the
    clover term is switched off."""
    dims = (4, 4, 4, 4)
    op = O.Operator(dims, I.gauge_exp(dims, 0.5, 44), 0.12, 1.0)
    rd = op.rounded()
    assert np.array_equal(rd.U, O.round_half(op.U)) and np.array_equal(rd.A, O.round_half(op.clover_matrix()))
    assert np.array_equal(rd.U.real, op.U.real.astype(np.float32).astype(np.float16).astype(np.float64))
    psi, chi = I.spinor(dims, 45), I.spinor(dims, 46)
    d = rel(rd.apply_D(psi), op.apply_D(psi))
    assert 1e-5 < d < 5e-4                                    # 2^-11 = 4.9e-4 per entry at most
    g5 = np.array([1, 1, -1, -1])[None, :, None]
    lhs = np.vdot(chi, g5 * rd.apply_D(psi))
    rhs = np.conj(np.vdot(psi, g5 * rd.apply_D(chi)))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # kappa-independent check of the link part: with A = 1 the explicit operator is D[round(U), c_sw = 0]
    one = np.zeros((op.V, 12, 12), complex) + np.eye(12)
    hop = op.with_operands(O.round_half(op.U), one)
    ref = O.Operator(dims, O.round_half(op.U), 0.12, 0.0)      # c_sw = 0: no clover term, links used as given
    assert rel(hop.apply_D(psi), ref.apply_D(psi)) < 1e-15
    # K_RAS of the rounded operator differs from the exact one at the rounding level, not more
    k0 = op.ras_apply((2, 2, 2, 2), 0, 2, 3, psi)
    k1 = rd.ras_apply((2, 2, 2, 2), 0, 2, 3, psi)
    assert 1e-5 < rel(k1, k0) < 2e-3
