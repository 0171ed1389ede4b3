"""Pins for the oracle's gamma algebra, operator M, solve and covariant derivative.

None of these re-types the oracle's formula against itself: they use algebraic identities,
momentum-space closed forms, gauge covariance, and an independently assembled dense matrix
(tests/dense_ref.py) with numpy LU.  [B:ns] = BASELINE.json north_star.
"""
import numpy as np
import pytest

import dense_ref as dr
from paper_1401_6750_b200 import inputs

C1 = inputs.CONFIGS["c1"]


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ------------------------------------------------------------------ gamma algebra
def test_gamma_clifford_hermitian(orc):
    g = [orc.gamma(m) for m in range(4)]
    for m in range(4):
        assert np.allclose(g[m], g[m].conj().T)
        for n in range(4):
            assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2.0 * (m == n) * np.eye(4))
    g5 = orc.gamma(4)
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))


def test_gamma_matches_pauli_kron(orc):
    for m in range(4):
        assert np.allclose(orc.gamma(m), dr.GAMMA[m])


def test_Gamma16_basis(orc):
    G = np.array([orc.Gamma(n) for n in range(16)])
    assert np.linalg.matrix_rank(G.reshape(16, 16)) == 16
    assert np.allclose(G[0], np.eye(4))
    assert np.allclose(G[15], orc.gamma(4))
    for n in range(16):
        assert np.allclose(G[n], dr.big_gamma(n))
        # signed / phased permutation matrices: one nonzero of modulus 1 per row
        assert np.allclose(np.sort(np.abs(G[n]), axis=1)[:, :3], 0)
        assert np.allclose(np.abs(G[n]).sum(axis=1), 1)


# ------------------------------------------------------------------ operator identities
@pytest.mark.parametrize("tb", [-1, 1])
def test_gamma5_hermiticity(orc, tb):
    """gamma5 M(mu) gamma5 = M(-mu)^dag  [B:ns]."""
    dims = (4, 2, 2, 4)
    U = inputs.gauge_field(dims, 0.3, 11)
    phi = inputs.random_spinor(dims, 12)
    psi = inputs.random_spinor(dims, 13)
    g5 = np.array([1, 1, -1, -1]).reshape(4, 1)
    k, mu = 0.156, 0.05
    lhs = vdot(phi, g5 * orc.apply_M(g5 * psi, U, k, mu, tb))
    rhs = vdot(orc.apply_M(phi, U, k, -mu, tb), psi)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    # and the explicitly written dagger is the adjoint
    lhs2 = vdot(phi, orc.apply_M(psi, U, k, mu, tb))
    rhs2 = vdot(orc.apply_M(phi, U, k, mu, tb, dagger=True), psi)
    assert abs(lhs2 - rhs2) < 1e-12 * abs(lhs2)
    # a wrong-sign twist would pass hermiticity with mu -> mu: make sure mu matters
    assert abs(vdot(orc.apply_M(phi, U, k, mu, tb), psi) - rhs) > 1e-6 * abs(rhs)


@pytest.mark.parametrize("tb", [-1, 1])
def test_free_field_plane_waves(orc, tb):
    """U = 1: M u e^{ipx} = Mtilde(p) u e^{ipx},
    Mtilde = 1 + 2 i kappa mu g5 - 2 kappa sum_mu (cos p_mu - i g_mu sin p_mu); p_t = 2pi(n+1/2)/T if tb=-1."""
    dims = (4, 6, 2, 8)
    lx, ly, lz, lt = dims
    U = inputs.unit_gauge(dims)
    k, mu = 0.12, 0.07
    rng = np.random.default_rng(5)
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    for n in [(1, 2, 0, 3), (3, 5, 1, 0), (0, 0, 0, 0)]:
        p = np.array([2 * np.pi * n[0] / lx, 2 * np.pi * n[1] / ly, 2 * np.pi * n[2] / lz,
                      2 * np.pi * (n[3] + (0.5 if tb == -1 else 0.0)) / lt])
        u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        wave = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
        psi = wave[..., None, None] * u
        Mt = np.eye(4) + 2j * k * mu * dr.GAMMA5
        for m in range(4):
            Mt = Mt - 2 * k * (np.cos(p[m]) * np.eye(4) - 1j * np.sin(p[m]) * dr.GAMMA[m])
        want = wave[..., None, None] * (Mt @ u)
        got = orc.apply_M(psi, U, k, mu, tb)
        assert np.allclose(got, want, atol=1e-13)
        wantd = wave[..., None, None] * (Mt.conj().T @ u)
        assert np.allclose(orc.apply_M(psi, U, k, mu, tb, dagger=True), wantd, atol=1e-13)


def test_constant_mode_value(orc):
    """mu = 0, U = 1, periodic, constant spinor: M = 1 - 8 kappa."""
    dims = (2, 2, 4, 2)
    psi = np.ones((2, 4, 2, 2, 4, 3), dtype=complex)
    out = orc.apply_M(psi, inputs.unit_gauge(dims), 0.1, 0.0, tb=1)
    assert np.allclose(out, (1 - 0.8) * psi)


def gauge_transform(U, g):
    """U^g_mu(x) = g(x) U_mu(x) g^dag(x+mu)."""
    out = np.empty_like(U)
    for m, ax in enumerate([3, 2, 1, 0]):
        gp = np.roll(g, -1, axis=ax)
        out[..., m, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, U[..., m, :, :], gp.conj())
    return out


@pytest.mark.parametrize("tb", [-1, 1])
def test_gauge_covariance(orc, tb):
    """M[U^g](g psi) = g M[U] psi  [B:ns]."""
    dims = (4, 4, 2, 4)
    U = inputs.gauge_field(dims, 0.3, 21)
    g = inputs.random_su3_field(dims, 22)
    psi = inputs.random_spinor(dims, 23)
    gpsi = np.einsum("...ab,...sb->...sa", g, psi)
    lhs = orc.apply_M(gpsi, gauge_transform(U, g), 0.15, 0.02, tb)
    rhs = np.einsum("...ab,...sb->...sa", g, orc.apply_M(psi, U, 0.15, 0.02, tb))
    assert np.linalg.norm(lhs - rhs) < 1e-13 * np.linalg.norm(rhs)


@pytest.mark.parametrize("dims,tb", [((2, 2, 2, 2), -1), ((2, 2, 2, 2), 1), ((4, 2, 2, 4), -1)])
def test_dense_matrix(orc, dims, tb):
    """oracle apply_M / apply_Mdag vs independently assembled dense matrix (2^4: fwd/bwd hops
    land on the same neighbour and add)  [B:ns]."""
    U = inputs.gauge_field(dims, 0.3, 31)
    k, mu = 0.156, 0.01
    M = dr.dense_M(U, dims, k, mu, tb)
    psi = inputs.random_spinor(dims, 32)
    want = (M @ psi.ravel()).reshape(psi.shape)
    assert np.linalg.norm(orc.apply_M(psi, U, k, mu, tb) - want) < 1e-13 * np.linalg.norm(want)
    wantd = (M.conj().T @ psi.ravel()).reshape(psi.shape)
    assert np.linalg.norm(orc.apply_M(psi, U, k, mu, tb, dagger=True) - wantd) < 1e-13 * np.linalg.norm(wantd)


# ------------------------------------------------------------------ solve
def test_solve_vs_dense_lu(orc):
    """brute-force dense inversion of M on 2^4  [B:ns]."""
    dims = (2, 2, 2, 2)
    U = inputs.gauge_field(dims, 0.3, 41)
    eta = inputs.z4_source(dims, 42, 0)
    k, mu = 0.156, 0.01
    s, it, tr, st = orc.solve(eta, U, k, mu, 1e-12)
    want = np.linalg.solve(dr.dense_M(U, dims, k, mu, -1), eta.ravel()).reshape(eta.shape)
    assert st == 0 and tr <= 1e-12
    assert np.linalg.norm(s - want) < 1e-10 * np.linalg.norm(want)


def test_solve_c1_residuals(orc):
    """config c1: rho = 1e-10 reached; LP stop is the first iterate with true residual <= rho."""
    dims = C1["dims"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    eta = inputs.z4_source(dims, C1["src_seed"], 0)
    s, it, tr, st = orc.solve(eta, U, C1["kappa"], C1["mu"], 1e-10)
    assert st == 0 and tr <= 1.0001e-10 and 20 < it < 400
    r = np.linalg.norm(eta - orc.apply_M(s, U, C1["kappa"], C1["mu"])) / np.linalg.norm(eta)
    assert abs(r - tr) < 1e-14
    assert abs(orc.true_residual(s, eta, U, C1["kappa"], C1["mu"]) - tr) < 1e-14
    s2, it2, tr2, st2 = orc.solve(eta, U, C1["kappa"], C1["mu"], 1e-2)
    assert st2 == 0 and tr2 <= 1e-2 and it2 < it
    # max_iter hit is reported
    _, it3, tr3, st3 = orc.solve(eta, U, C1["kappa"], C1["mu"], 1e-10, max_iter=3)
    assert st3 == 1 and it3 == 3 and tr3 > 1e-10


# ------------------------------------------------------------------ covariant derivative
def test_cov_deriv_plane_wave(orc):
    """U = 1: D_mu e^{ipx} = i sin(p_mu) e^{ipx}."""
    dims = (4, 6, 2, 8)
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    p = np.array([2 * np.pi * 1 / lx, 2 * np.pi * 2 / ly, 2 * np.pi * 1 / lz, 2 * np.pi * 3.5 / lt])
    u = np.arange(12).reshape(4, 3) + 1j
    psi = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))[..., None, None] * u
    for m in range(4):
        got = orc.cov_deriv(psi, inputs.unit_gauge(dims), m, tb=-1)
        assert np.allclose(got, 1j * np.sin(p[m]) * psi, atol=1e-13)


@pytest.mark.parametrize("tb", [-1, 1])
def test_cov_deriv_dense_antihermitian_covariant(orc, tb):
    dims = (2, 4, 2, 4)
    U = inputs.gauge_field(dims, 0.3, 51)
    psi = inputs.random_spinor(dims, 52)
    phi = inputs.random_spinor(dims, 53)
    g = inputs.random_su3_field(dims, 54)
    for m in range(4):
        D = dr.dense_cov_deriv(U, dims, m, tb)
        got = orc.cov_deriv(psi, U, m, tb)
        assert np.allclose(got.ravel(), D @ psi.ravel(), atol=1e-13)
        # anti-Hermitian: <phi, D psi> = -<D phi, psi>  (summation by parts)
        a = vdot(phi, got)
        b = vdot(orc.cov_deriv(phi, U, m, tb), psi)
        assert abs(a + b) < 1e-12 * abs(a)
        gpsi = np.einsum("...ab,...sb->...sa", g, psi)
        lhs = orc.cov_deriv(gpsi, gauge_transform(U, g), m, tb)
        rhs = np.einsum("...ab,...sb->...sa", g, got)
        assert np.linalg.norm(lhs - rhs) < 1e-13 * np.linalg.norm(rhs)
