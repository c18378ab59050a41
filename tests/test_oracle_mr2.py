"""Pins of the oracle's stronger block solver (wco_mr2_block: restarted two-dimensional minimal residual = GMRES(2);
SURVEY.md 8(f) NEXT-4, reading R2) against things that do not come from the oracle: numpy least squares on the
dense restricted operator, the closed-form free-field symbol (minimal polynomial of degree 2), and the defining
minimisation property."""
import numpy as np
import pytest

import oracle as O
from paper_1011_3318_b200 import inputs as I
from test_oracle_operator import TG, coords
from test_oracle_solver import box_sites, dense_from, dense_S


@pytest.fixture(scope="module")
def small():
    dims = (6, 4, 2, 2)
    U = I.gauge_exp(dims, 0.5, 7)
    op = O.Operator(dims, U, 0.12, 1.0)
    D = dense_from(op.apply_D, 12 * op.V)
    return dims, op, D


def lstsq_cycle(Dl, rho):
    """One cycle written out with numpy: minimise |rho - Dl K c| over K = [rho, Dl rho]."""
    K = np.stack([rho, Dl @ rho], axis=1)
    c = np.linalg.lstsq(Dl @ K, rho, rcond=None)[0]
    dv = K @ c
    return dv, rho - Dl @ dv


@pytest.mark.parametrize("s", [0, 1])
def test_mr2_is_dense_least_squares(small, s):
    dims, op, D = small
    block = (2, 2, 2, 2)
    origin, start, ext = op.domain_box(block, s, 2)
    sites = box_sites(dims, start, ext)
    comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
    Dl = D[np.ix_(comp, comp)]
    r = I.spinor(dims, 9)
    rl = r.reshape(-1)[comp]
    v_want, rho_want = np.zeros_like(rl), rl.copy()
    for cyc in range(1, 4):
        dv, rho_want = lstsq_cycle(Dl, rho_want)
        v_want = v_want + dv
        v, rho = op.mr2_block(start, ext, 2 * cyc, r)
        assert np.abs(v.reshape(-1) - v_want).max() < 1e-12
        assert np.abs(rho.reshape(-1) - rho_want).max() < 1e-12
        assert np.abs(rho.reshape(-1) - (rl - Dl @ v.reshape(-1))).max() < 1e-13
        # the new residual is orthogonal to both directions of the cycle
        if cyc == 1:
            for qk in (Dl @ rl, Dl @ (Dl @ rl)):
                assert abs(np.vdot(qk, rho.reshape(-1))) < 1e-12 * np.linalg.norm(qk) * np.linalg.norm(rl)
    # odd count: the pairs, then one plain MR iteration
    v3, rho3 = op.mr2_block(start, ext, 3, r)
    dv, rho2 = lstsq_cycle(Dl, rl)
    q = Dl @ rho2
    a = np.vdot(q, rho2) / np.vdot(q, q)
    assert np.abs(v3.reshape(-1) - (dv + a * rho2)).max() < 1e-12
    assert np.abs(rho3.reshape(-1) - (rho2 - a * q)).max() < 1e-12
    # degenerate cases: zero iterations, zero residual (no NaN)
    v0, rho0 = op.mr2_block(start, ext, 0, r)
    assert np.abs(v0).max() == 0 and np.array_equal(rho0.reshape(-1), rl)
    z, _ = op.mr2_block(start, ext, 4, np.zeros_like(r))
    assert np.abs(z).max() == 0


@pytest.mark.parametrize("s", [0, 1])
def test_mr2_never_worse_than_two_mr_steps(small, s):
    """span{rho, D rho} contains what two MR steps can reach from rho, so a cycle cannot leave a larger residual."""
    dims, op, D = small
    origin, start, ext = op.domain_box((2, 2, 2, 2), s, 0)
    r = I.spinor(dims, 10)
    for n in (2, 4, 6, 8):
        _, rho_mr = op.mr_block(start, ext, n, r)
        _, rho_2 = op.mr2_block(start, ext, n, r)
        assert np.linalg.norm(rho_2) <= np.linalg.norm(rho_mr) * (1 + 1e-14)
    assert np.linalg.norm(op.mr2_block(start, ext, 8, r)[1]) < 0.9 * np.linalg.norm(op.mr_block(start, ext, 8, r)[1])


def test_mr2_solves_free_field_plane_wave_in_one_cycle():
    """U = 1, one domain = the whole lattice (wrap-around hops kept, reading Q7): on psi = u e^{ipx} D is the 4x4 symbol
    D(p) = a + 2 i kappa sum_mu sin(p_mu) gamma_mu, whose square is a scalar, so its minimal polynomial has degree 2 and
    one cycle returns D^-1 r for ANY u; two MR steps do not."""
    dims = (4, 6, 4, 4)
    kappa = 0.12
    op = O.Operator(dims, I.gauge_unit(dims), kappa, 1.3)
    xs = coords(dims)
    rng = np.random.default_rng(11)
    p = 2 * np.pi * np.array((1, 2, 3, 1)) / np.array(dims)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    r = np.exp(1j * (xs @ p))[:, None, None] * u[None]
    sym = (1 - 2 * kappa * np.cos(p).sum()) * np.eye(4) + 2j * kappa * sum(np.sin(p[m]) * TG[m] for m in range(4))
    want = np.exp(1j * (xs @ p))[:, None, None] * np.linalg.solve(sym, u)[None]
    v, rho = op.mr2_block((0, 0, 0, 0), dims, 2, r)
    assert np.linalg.norm(rho) < 1e-11 * np.linalg.norm(r)  # normal equations: rounding times the condition of the 2x2 Gram matrix
    assert np.abs(v - want).max() < 1e-11
    _, rho_mr = op.mr_block((0, 0, 0, 0), dims, 2, r)
    assert np.linalg.norm(rho_mr) > 1e-4 * np.linalg.norm(r)
    # an eigenvector of D: q2 is parallel to q1, the determinant vanishes and the cycle falls back to the exact MR step
    lam, vec = np.linalg.eig(sym)
    r1 = np.exp(1j * (xs @ p))[:, None, None] * np.outer(vec[:, 0], [1.0, 0.5j, -2.0])[None]
    v1, rho1 = op.mr2_block((0, 0, 0, 0), dims, 2, r1)
    assert np.all(np.isfinite(v1)) and np.linalg.norm(rho1) < 1e-12 * np.linalg.norm(r1)
    assert np.abs(v1 - r1 / lam[0]).max() < 1e-12


def test_mr2_is_scale_invariant(small):
    """The block solve is linear in the scale of its input: a residual of norm 1e-120 (squared norms 1e-240, whose PRODUCT
    would underflow) gives the scaled result, not the degenerate-pair fallback (reading R2: the 2x2 solve is
    written without a product of two squared norms)."""
    dims, op, D = small
    origin, start, ext = op.domain_box((2, 2, 2, 2), 1, 3)
    r = I.spinor(dims, 13)
    v, rho = op.mr2_block(start, ext, 4, r)
    v2, rho2 = op.mr2_block(start, ext, 4, 1e-120 * r)
    assert np.abs(v2 * 1e120 - v).max() < 1e-12 * np.abs(v).max()
    assert np.abs(rho2 * 1e120 - rho).max() < 1e-12 * np.abs(rho).max()
    assert np.abs(v - op.mr_block(start, ext, 4, r)[0]).max() > 1e-3   # and it is not the MR fallback


@pytest.mark.parametrize("s,nras", [(0, 1), (0, 3), (1, 2)])
def test_alg1_with_mr2_blocks(small, s, nras):
    """Alg. 1 with the block solver switched (wco_set_block_solver through Operator.with_block_solver): every cycle is the
    disjoint sum of the restricted block solutions, written out here with mr2_block and the dense D."""
    dims, op, D = small
    block = (2, 2, 2, 2)
    eta = I.spinor(dims, 12)
    got = op.with_block_solver("mr2").ras_apply(block, s, 4, nras, eta)
    phi = np.zeros(12 * op.V, complex)
    r = eta.reshape(-1).copy()
    for j in range(nras):
        v = np.zeros_like(phi)
        for idx in range(op.domain_count(block)):
            origin, start, ext = op.domain_box(block, s, idx)
            sites = box_sites(dims, start, ext)
            vl, _ = op.mr2_block(start, ext, 4, r.reshape(-1, 4, 3))
            pos = {g: k for k, g in enumerate(sites)}
            for g in box_sites(dims, origin, block):
                v[12 * g:12 * g + 12] = vl.reshape(-1, 12)[pos[g]]
        phi += v
        r -= D @ v
    assert np.abs(got.reshape(-1) - phi).max() < 1e-12
    # the switch does not leak: the plain operator still runs MR
    a = op.ras_apply(block, s, 4, nras, eta)
    assert np.abs(a - got).max() > 1e-6
    # many cycles of exact-enough block solves converge to Eq. (2.1) with exact block inverses
    S = dense_S(dims, op, D, block, s)
    far = op.with_block_solver("mr2").ras_apply(block, s, 200, 1, eta)
    assert np.abs(far.reshape(-1) - S @ eta.reshape(-1)).max() < 1e-10
