"""Pins for the oracle's restricted operator, MR block solve, RAS iteration (Alg. 1) and BiCGStab.
CPU only.  Dense matrices are obtained column by column from the (already pinned) oracle apply_D and
then handled by numpy/LAPACK, i.e. by something other than the routine under test.
"""
import numpy as np
import pytest

import oracle as O
from paper_1011_3318_b200 import inputs as I
from test_oracle_operator import coords, gauge_transform


def dense_from(apply, n):
    M = np.empty((n, n), complex)
    e = np.zeros(n, complex)
    for k in range(n):
        e[k] = 1
        M[:, k] = apply(e.reshape(-1, 4, 3)).reshape(-1)
        e[k] = 0
    return M


def box_sites(dims, start, ext):
    """Global site indices of the box, local lexicographic order (x fastest) -- written independently here."""
    out = []
    for ct in range(ext[3]):
        for cz in range(ext[2]):
            for cy in range(ext[1]):
                for cx in range(ext[0]):
                    x = [(start[m] + c) % dims[m] for m, c in enumerate((cx, cy, cz, ct))]
                    out.append(x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3])))
    return np.array(out)


@pytest.fixture(scope="module")
def small():
    dims = (6, 4, 2, 2)
    U = I.gauge_exp(dims, 0.5, 7)
    op = O.Operator(dims, U, 0.12, 1.0)
    D = dense_from(op.apply_D, 12 * op.V)
    return dims, op, D


def test_dense_LU_2to4():
    """north_star self-check 4: dense LU on a 2^4 lattice (192 x 192) vs the iterative solvers.
    L = 2: forward and backward neighbour coincide and both hops are added (reading Q19)."""
    dims = (2, 2, 2, 2)
    op = O.Operator(dims, I.gauge_exp(dims, 0.5, 1), 0.12, 1.0)
    D = dense_from(op.apply_D, 192)
    # 8 hops + site term: 9 distinct 3x3-colour blocks would need L>2; at L=2 fwd/bwd merge
    eta = I.spinor(dims, 1)
    want = np.linalg.solve(D, eta.reshape(-1))
    x, info = op.bicgstab(eta, tol=1e-13)
    assert info["status"] == 0 and info["rel_resid_true"] < 1e-12
    assert np.abs(x.reshape(-1) - want).max() < 1e-11
    x, info = op.nested_bicgstab(eta, tol=1e-13, inner_tol=1e-4)
    assert info["status"] == 0 and info["rel_resid_true"] < 1e-13
    assert np.abs(x.reshape(-1) - want).max() < 1e-11
    x, info = op.bicgstab(eta, tol=1e-13, ras=dict(domain=(2, 2, 1, 1), overlap=0, block_iters=3, nras=2))
    assert info["status"] == 0 and np.abs(x.reshape(-1) - want).max() < 1e-11
    assert abs(op.true_residual(eta, want.reshape(-1, 4, 3))) < 1e-14


@pytest.mark.parametrize("s", [0, 1])
def test_restricted_operator_is_principal_submatrix(small, s):
    """D_Omega' = principal sub-matrix of D on Omega' (reading Q7).  With s = 1 the y extent
    b+2s = 4 = L_y covers the direction, so its wrap-around hops stay inside and are kept."""
    dims, op, D = small
    block = (2, 2, 2, 2)
    nd = op.domain_count(block)
    assert nd == 6
    for idx in (0, 2, 5):
        origin, start, ext = op.domain_box(block, s, idx)
        assert ext == ((2 + 2 * s, 2 + 2 * s, 2, 2))
        sites = box_sites(dims, start, ext)
        assert len(set(sites)) == len(sites)
        comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
        want = np.zeros_like(D)
        want[np.ix_(comp, comp)] = D[np.ix_(comp, comp)]
        got = dense_from(lambda v: op.apply_D_restricted(block, s, idx, v), 12 * op.V)
        assert np.abs(got - want).max() < 1e-15


def test_restricted_whole_lattice_is_D(small):
    dims, op, D = small
    psi = I.spinor(dims, 3)
    assert np.array_equal(op.apply_D_restricted(dims, 0, 0, psi), op.apply_D(psi))
    assert np.array_equal(op.apply_D_restricted(dims, 2, 0, psi), op.apply_D(psi))  # unsplit dirs not extended


def test_invalid_decompositions(small):
    dims, op, _ = small
    with pytest.raises(ValueError):
        op.domain_box((4, 4, 2, 2), 0, 0)  # 4 does not divide 6
    with pytest.raises(ValueError):
        op.domain_box((2, 2, 2, 2), 2, 0)  # b+2s = 6 > L_y = 4
    with pytest.raises(ValueError):
        op.ras_apply((2, 2, 2, 2), 2, 1, 1, I.spinor(dims, 1))


@pytest.mark.parametrize("s", [0, 1])
def test_mr_properties(small, s):
    """MR: |rho| non-increasing, <q, rho_new> = 0 after each step, rho = r - D_Omega' v, and many
    iterations reproduce the dense block inverse (SURVEY 8(c) pins; reading Q9)."""
    dims, op, D = small
    block = (2, 2, 2, 2)
    origin, start, ext = op.domain_box(block, s, 1)
    sites = box_sites(dims, start, ext)
    comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
    Dl = D[np.ix_(comp, comp)]
    r = I.spinor(dims, 5)
    rl = r.reshape(-1)[comp]
    prev = np.linalg.norm(rl)
    rho_prev = rl
    for n in range(1, 7):
        v, rho = op.mr_block(start, ext, n, r)
        v, rho = v.reshape(-1), rho.reshape(-1)
        assert np.abs(rho - (rl - Dl @ v)).max() < 1e-13
        q = Dl @ rho_prev
        assert abs(np.vdot(q, rho)) < 1e-12 * np.linalg.norm(q) * np.linalg.norm(rho_prev)
        nr = np.linalg.norm(rho)
        assert nr <= prev * (1 + 1e-15)
        prev, rho_prev = nr, rho
    # first step in closed form
    v1, _ = op.mr_block(start, ext, 1, r)
    q = Dl @ rl
    assert np.abs(v1.reshape(-1) - (np.vdot(q, rl) / np.vdot(q, q)) * rl).max() < 1e-14
    vN, _ = op.mr_block(start, ext, 300, r)
    assert np.abs(vN.reshape(-1) - np.linalg.solve(Dl, rl)).max() < 1e-11
    v0, rho0 = op.mr_block(start, ext, 0, r)
    assert np.abs(v0).max() == 0 and np.array_equal(rho0.reshape(-1), rl)
    # zero residual in a domain: alpha := 0, no NaN
    z, _ = op.mr_block(start, ext, 3, np.zeros_like(r))
    assert np.abs(z).max() == 0


def dense_S(dims, op, D, block, s):
    """S = sum_i R_i^T-placed (D_Omega'_i)^-1 P_Omega'_i of Eq. (2.1), dense, with exact block inverses."""
    n = D.shape[0]
    S = np.zeros((n, n), complex)
    owner = np.zeros(op.V, int)
    for idx in range(op.domain_count(block)):
        origin, start, ext = op.domain_box(block, s, idx)
        sites = box_sites(dims, start, ext)
        comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
        inv = np.linalg.inv(D[np.ix_(comp, comp)])
        bulk = box_sites(dims, origin, block)
        owner[bulk] += 1
        pos = {g: k for k, g in enumerate(sites)}
        rows_l = (12 * np.array([pos[g] for g in bulk])[:, None] + np.arange(12)[None]).reshape(-1)
        rows_g = (12 * bulk[:, None] + np.arange(12)[None]).reshape(-1)
        S[np.ix_(rows_g, comp)] += inv[rows_l, :]
    assert np.all(owner == 1)  # partition of unity: every site restricted-to by exactly one domain
    return S


@pytest.mark.parametrize("s,nras", [(0, 1), (0, 3), (1, 1), (1, 3)])
def test_alg1_equals_eq21(small, s, nras):
    """Alg. 1 == K_RAS = S sum_{j<NRAS} (1 - D S)^j  (Eq. 2.1) when the
    block solve is exact (MR run to convergence)."""
    dims, op, D = small
    block = (2, 2, 2, 2)
    S = dense_S(dims, op, D, block, s)
    n = D.shape[0]
    K = np.zeros((n, n), complex)
    T = np.eye(n, dtype=complex)
    for _ in range(nras):
        K += S @ T
        T = (np.eye(n) - D @ S) @ T
    eta = I.spinor(dims, 8)
    got = op.ras_apply(block, s, 400, nras, eta).reshape(-1)
    want = K @ eta.reshape(-1)
    assert np.abs(got - want).max() < 1e-10 * np.abs(want).max()
    if s == 0:  # block-Jacobi: S is block diagonal
        origin, start, ext = op.domain_box(block, 0, 0)
        sites = box_sites(dims, start, ext)
        comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
        rest = np.setdiff1d(np.arange(n), comp)
        assert np.abs(S[np.ix_(comp, rest)]).max() == 0


@pytest.mark.parametrize("ncycle", [1, 2])
def test_sap_equals_block_gauss_seidel(small, ncycle):
    """Multiplicative Schwarz (SAP, PAPER.md:33 ref [5]) with exact block solves == the dense
    red-black block Gauss-Seidel iteration phi += S_c r, r -= D S_c r over the colours c = 0, 1; a black half step
    leaves a zero residual on the black domains; and SAP reduces the residual further than RAS with the same number
    of cycles."""
    dims = (4, 4, 2, 2)  # 2 x 2 x 1 x 1 blocks: even in every cut direction
    op = O.Operator(dims, I.gauge_exp(dims, 0.5, 7), 0.12, 1.0)
    D = dense_from(op.apply_D, 12 * op.V)
    block = (2, 2, 2, 2)
    n = D.shape[0]
    nblk = [dims[mu] // block[mu] for mu in range(4)]
    Sc = [np.zeros((n, n), complex), np.zeros((n, n), complex)]
    comps = [[], []]
    for idx in range(op.domain_count(block)):
        bc, par = idx, 0
        for mu in range(4):
            par += bc % nblk[mu]
            bc //= nblk[mu]
        origin, start, ext = op.domain_box(block, 0, idx)
        sites = box_sites(dims, start, ext)
        comp = (12 * sites[:, None] + np.arange(12)[None]).reshape(-1)
        Sc[par & 1][np.ix_(comp, comp)] = np.linalg.inv(D[np.ix_(comp, comp)])
        comps[par & 1].append(comp)
    eta = I.spinor(dims, 8)
    r = eta.reshape(-1).copy()
    phi = np.zeros(n, complex)
    for cyc in range(ncycle):
        for c in (0, 1):
            v = Sc[c] @ r
            phi += v
            r = r - D @ v
            assert np.abs(r[np.concatenate(comps[c])]).max() < 1e-12   # exact solve: residual vanishes there
    got = op.sap_apply(block, 400, ncycle, eta).reshape(-1)
    assert np.abs(got - phi).max() < 1e-10 * np.abs(phi).max()
    res_sap = np.linalg.norm(eta.reshape(-1) - D @ got)
    ras = op.ras_apply(block, 0, 400, ncycle, eta).reshape(-1)
    assert res_sap < np.linalg.norm(eta.reshape(-1) - D @ ras)


def test_sap_needs_two_colourable_decomposition(small):
    dims, op, D = small
    with pytest.raises(ValueError):
        op.sap_apply(dims, 3, 1, I.spinor(dims, 1))           # a single domain cannot be coloured
    with pytest.raises(ValueError):
        op.sap_apply((2, 2, 2, 2), 3, 1, I.spinor(dims, 1))   # 3 blocks in x: neighbours across the wrap share a colour


def test_ras_single_domain_is_inverse(small):
    """north_star self-check 5: one domain covering the whole lattice + exact block solve => phi = D^-1 eta."""
    dims, op, D = small
    eta = I.spinor(dims, 2)
    phi = op.ras_apply(dims, 0, 400, 1, eta)
    want = np.linalg.solve(D, eta.reshape(-1))
    assert np.abs(phi.reshape(-1) - want).max() < 1e-11
    assert op.true_residual(eta, phi) < 1e-12


@pytest.mark.parametrize("s", [0, 1])
def test_ras_identity_operator_partition_of_unity(s):
    """kappa = 0 => D = 1, MR is exact after one step, so K_RAS r = r for any decomposition and overlap:
    every site is written exactly once by the restriction."""
    dims = (6, 4, 4, 2)
    op = O.Operator(dims, I.gauge_exp(dims, 0.5, 1), 0.0, 1.0)
    r = I.spinor(dims, 3)
    out = op.ras_apply((2, 2, 2, 2), s, 1, 1, r)
    assert np.abs(out - r).max() < 1e-15
    out = op.ras_apply((2, 2, 2, 2), s, 2, 3, r)  # r - Dv = 0 after the first cycle
    assert np.abs(out - r).max() < 1e-15


def test_ras_one_mr_step_is_neumann_like(small):
    """NRAS cycles telescoping: phi_NRAS = sum_j S_j r_j with r_{j+1} = r_j - D S_j r_j.  Checked by chaining
    NRAS = 1 applications by hand through apply_D."""
    dims, op, D = small
    block, s, nit = (2, 2, 2, 2), 1, 3
    eta = I.spinor(dims, 6)
    r = eta.copy()
    phi = np.zeros_like(eta)
    for j in range(3):
        v = op.ras_apply(block, s, nit, 1, r)
        phi += v
        r = r - op.apply_D(v)
    got = op.ras_apply(block, s, nit, 3, eta)
    assert np.abs(got - phi).max() < 1e-13


def test_bicgstab_and_covariance():
    """Solution covariance phi[U^g, g eta] = g phi[U, eta] (north_star self-check 3) + true residuals."""
    dims = (4, 4, 4, 4)
    U = I.gauge_exp(dims, 0.5, 1)
    g = I.su3_field(dims, 21)
    eta = I.spinor(dims, 1)
    ras = dict(domain=(2, 2, 2, 2), overlap=0, block_iters=4, nras=1)
    op, opg = O.Operator(dims, U, 0.12, 1.0), O.Operator(dims, gauge_transform(dims, U, g), 0.12, 1.0)
    geta = np.einsum("vab,vsb->vsa", g, eta)
    for kw in (dict(), dict(ras=ras)):
        x, info = op.bicgstab(eta, tol=1e-13, **kw)
        xg, infog = opg.bicgstab(geta, tol=1e-13, **kw)
        assert info["status"] == 0 and infog["status"] == 0
        assert info["rel_resid_true"] < 2e-13 and infog["rel_resid_true"] < 2e-13
        assert np.abs(xg - np.einsum("vab,vsb->vsa", g, x)).max() < 1e-11
    x0, i0 = op.bicgstab(eta, tol=1e-12)
    x1, i1 = op.bicgstab(eta, tol=1e-12, ras=ras)
    assert i1["iters"] < i0["iters"]  # RAS reduces the iteration count
    assert i1["dv"] == 2 * i1["iters"] or i1["dv"] == 2 * i1["iters"] - 1
    x2, i2 = op.nested_bicgstab(eta, tol=1e-12, inner_tol=1e-5, ras=ras)
    assert i2["status"] == 0 and i2["rel_resid_true"] <= 1e-12
    assert np.abs(x2 - x0).max() < 1e-10
