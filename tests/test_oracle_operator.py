"""Pins for the oracle's operator part (oracle/wcoracle.c): gamma algebra, hopping term, clover term,
gamma5-hermiticity, gauge covariance.  CPU only.  Every check is against something the oracle does not
compute itself: closed forms, algebraic identities, symmetry transformations built here with numpy.
"""
import itertools
import os

import numpy as np
import pytest

import oracle as O
from paper_1011_3318_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")

# The test's own gamma matrices, built from Pauli matrices by Kronecker products (chiral basis, reading Q2):
# gamma_k = sigma_2 (x) sigma_k  (k = x,y,z),  gamma_t = sigma_1 (x) 1.
PAULI = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]], complex),
         np.array([[1, 0], [0, -1]], complex)]
S0 = np.eye(2, dtype=complex)
TG = [np.kron(PAULI[1], PAULI[k]) for k in range(3)] + [np.kron(PAULI[0], S0)]


def coords(dims):
    V = I.volume(dims)
    i = np.arange(V)
    x = i % dims[0]
    y = (i // dims[0]) % dims[1]
    z = (i // (dims[0] * dims[1])) % dims[2]
    t = i // (dims[0] * dims[1] * dims[2])
    return np.stack([x, y, z, t], axis=1)


def test_gamma_algebra():
    g = [O.gamma(m) for m in range(4)]
    for m in range(4):
        assert np.array_equal(g[m], TG[m]), "oracle gamma != sigma (x) sigma construction"
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(4):
            assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2 * (m == n) * np.eye(4))
        for sg in (+1, -1):
            assert np.linalg.matrix_rank(np.eye(4) + sg * g[m]) == 2
    g5 = O.gamma(4)
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])


def test_sigma_blocks():
    """sigma_mu_nu = (i/2)[gamma_mu,gamma_nu]: Hermitian, block diagonal, with the 2x2 blocks of reading Q3."""
    s1, s2, s3 = PAULI
    expect = {(0, 1): (-s3, -s3), (0, 2): (s2, s2), (0, 3): (s1, -s1),
              (1, 2): (-s1, -s1), (1, 3): (s2, -s2), (2, 3): (s3, -s3)}
    for (m, n), (up, lo) in expect.items():
        s = O.sigma(m, n)
        assert np.allclose(s, s.conj().T)
        assert np.allclose(s, 0.5j * (TG[m] @ TG[n] - TG[n] @ TG[m]))
        assert np.allclose(s[:2, :2], up) and np.allclose(s[2:, 2:], lo)
        assert np.allclose(s[:2, 2:], 0) and np.allclose(s[2:, :2], 0)


def test_golden_free_field_closed_form():
    for line in open(os.path.join(GOLD, "free_field.txt")):
        if line.startswith("#") or not line.strip():
            continue
        kappa, px, py, pz, pt, a, b = [float(t) for t in line.split()]
        p = np.array([px, py, pz, pt])
        Dp = np.eye(4, dtype=complex)
        for m in range(4):
            Dp = Dp - kappa * ((np.eye(4) - TG[m]) * np.exp(1j * p[m]) + (np.eye(4) + TG[m]) * np.exp(-1j * p[m]))
        ev = np.linalg.eigvals(Dp)
        assert np.allclose(ev.real, a, atol=2e-9)
        assert np.allclose(sorted(ev.imag), [-b, -b, b, b], atol=2e-9)


@pytest.mark.parametrize("csw", [0.0, 1.3])
def test_free_field_plane_wave(csw):
    """U = 1: D acts on psi = u e^{ipx} as the 4x4 symbol D(p) (x) 1_colour; clover term vanishes (F = 0)."""
    dims = (4, 6, 4, 8)  # distinct extents catch transposed indices
    kappa = 0.12
    op = O.Operator(dims, I.gauge_unit(dims), kappa, csw)
    assert np.abs(op.F).max() == 0.0
    xs = coords(dims)
    rng = np.random.default_rng(5)
    for n in [(1, 2, 3, 1), (0, 5, 1, 7), (3, 0, 2, 4)]:
        p = 2 * np.pi * np.array(n) / np.array(dims)
        u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        psi = np.exp(1j * (xs @ p))[:, None, None] * u[None]
        sym = (1 - 2 * kappa * np.cos(p).sum()) * np.eye(4) + 2j * kappa * sum(np.sin(p[m]) * TG[m] for m in range(4))
        want = np.exp(1j * (xs @ p))[:, None, None] * (sym @ u)[None]
        got = op.apply_D(psi)
        assert np.abs(got - want).max() < 1e-13
        # D^dag D symbol = |lambda|^2 for any u
        lam2 = (1 - 2 * kappa * np.cos(p).sum()) ** 2 + 4 * kappa ** 2 * (np.sin(p) ** 2).sum()
        assert np.allclose(np.vdot(got, got), lam2 * np.vdot(psi, psi))


@pytest.mark.parametrize("plane", range(6))
def test_field_strength_abelian(plane):
    """Constant abelian field U_nu(x) = exp(i phi x_mu): every (mu,nu) plaquette = e^{i phi}, so
    F_mu_nu = sin(phi) * 1 exactly and all other planes vanish; U_mu(x) = exp(i phi x_nu) gives -sin(phi).
    Pins the 1/8 normalisation, leaf orientation, index order and antisymmetry (reading Q4)."""
    planes = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    mu, nu = planes[plane]
    dims = (4, 6, 8, 4)
    xs = coords(dims)
    k = 1
    phi = 2 * np.pi * k / dims[mu]
    U = I.gauge_unit(dims)
    U[:, nu] = np.exp(1j * phi * xs[:, mu])[:, None, None] * np.eye(3)
    F = O.field_strength(dims, U)
    for q, _ in enumerate(planes):
        want = np.sin(phi) * np.eye(3) if q == plane else np.zeros((3, 3))
        assert np.abs(F[:, q] - want).max() < 1e-14
    phi2 = 2 * np.pi * k / dims[nu]
    U = I.gauge_unit(dims)
    U[:, mu] = np.exp(1j * phi2 * xs[:, nu])[:, None, None] * np.eye(3)
    F = O.field_strength(dims, U)
    assert np.abs(F[:, plane] + np.sin(phi2) * np.eye(3)).max() < 1e-14


def test_clover_matrix_closed_form():
    """On the abelian field the clover term is A = 1 - (c_sw kappa/2) sin(phi) sigma_mu_nu (x) 1_colour
    (north_star formula, literal coefficient: reading Q5).  D(c_sw) - D(0) isolates it."""
    dims = (4, 4, 6, 4)
    xs = coords(dims)
    kappa, csw = 0.11, 1.7
    psi = I.spinor(dims, 11)
    for (mu, nu) in [(0, 1), (1, 3), (2, 3)]:
        phi = 2 * np.pi / dims[mu]
        U = I.gauge_unit(dims)
        U[:, nu] = np.exp(1j * phi * xs[:, mu])[:, None, None] * np.eye(3)
        d1 = O.Operator(dims, U, kappa, csw).apply_D(psi)
        d0 = O.Operator(dims, U, kappa, 0.0).apply_D(psi)
        sig = 0.5j * (TG[mu] @ TG[nu] - TG[nu] @ TG[mu])
        want = -(csw * kappa / 2) * np.sin(phi) * np.einsum("ab,vbc->vac", sig, psi)
        assert np.abs((d1 - d0) - want).max() < 1e-14


def test_field_strength_hermitian_and_covariant():
    dims = (4, 4, 4, 4)
    U = I.gauge_exp(dims, 0.5, 1)
    F = O.field_strength(dims, U)
    assert np.abs(F - np.conj(np.swapaxes(F, 2, 3))).max() < 1e-15
    assert np.abs(F).max() > 0.05  # not trivially zero
    g = I.su3_field(dims, 3)
    Ug = gauge_transform(dims, U, g)
    Fg = O.field_strength(dims, Ug)
    want = np.einsum("vab,vpbc,vdc->vpad", g, F, np.conj(g))
    assert np.abs(Fg - want).max() < 1e-14


def gauge_transform(dims, U, g):
    """U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dag."""
    V = I.volume(dims)
    xs = coords(dims)
    out = np.empty_like(U)
    strides = np.array([1, dims[0], dims[0] * dims[1], dims[0] * dims[1] * dims[2]])
    for mu in range(4):
        y = xs.copy()
        y[:, mu] = (y[:, mu] + 1) % dims[mu]
        j = y @ strides
        out[:, mu] = np.einsum("vab,vbc,vdc->vad", g, U[:, mu], np.conj(g[j]))
    assert out.shape == (V, 4, 3, 3)
    return out


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 4, 6, 2)])
def test_gamma5_hermiticity(dims):
    """gamma5 D gamma5 = D^dagger:  <chi, g5 D psi> = conj <psi, g5 D chi>  (north_star self-check 1)."""
    U = I.gauge_exp(dims, 0.5, 1)
    op = O.Operator(dims, U, 0.12, 1.1)
    psi, chi = I.spinor(dims, 1, 0), I.spinor(dims, 1, 1)
    g5 = np.array([1, 1, -1, -1])[None, :, None]
    a = np.vdot(chi, g5 * op.apply_D(psi))
    b = np.vdot(psi, g5 * op.apply_D(chi))
    assert abs(a - np.conj(b)) < 1e-12 * abs(a)


@pytest.mark.parametrize("kind", ["exp", "haar"])
def test_gauge_covariance_of_D(kind):
    """D[U^g](g psi) = g D[U] psi (with clover)."""
    dims = (4, 2, 4, 6)
    U = I.gauge_exp(dims, 0.7, 3) if kind == "exp" else I.gauge_haar(dims, 4)
    g = I.su3_field(dims, 9)
    psi = I.spinor(dims, 2)
    op, opg = O.Operator(dims, U, 0.122, 1.2), O.Operator(dims, gauge_transform(dims, U, g), 0.122, 1.2)
    lhs = opg.apply_D(np.einsum("vab,vsb->vsa", g, psi))
    rhs = np.einsum("vab,vsb->vsa", g, op.apply_D(psi))
    assert np.abs(lhs - rhs).max() < 1e-13


def test_apply_D_sites_matches_full():
    dims = (4, 4, 4, 4)
    op = O.Operator(dims, I.gauge_haar(dims, 4), 0.1225, 1.0)
    psi = I.spinor(dims, 4)
    sites = np.array([0, 3, 17, 100, 255])
    assert np.array_equal(op.apply_D_sites(psi, sites), op.apply_D(psi)[sites])


def test_table1_consistency():
    rows = {}
    for line in open(os.path.join(GOLD, "table1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        rows[t[0]] = [float(v) for v in t[1:]]
    for c in range(4):
        assert abs(rows["copy_time"][c] - rows["t_dv_comm"][c] - rows["t_proj_comm"][c]) < 2e-3
        assert rows["total_time"][c] > rows["gpu_solver_time"][c] > rows["dv_time_total"][c]
    assert round(rows["total_time"][0] / rows["total_time"][1], 1) == 1.9  # "a factor two" PAPER.md:137
