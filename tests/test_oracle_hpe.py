"""Pins for the oracle's Hopping Parameter Expansion functions (reading 23).

PAPER.md:92: the interfaces compute "any ultra-local and one-derivative insertion with several variance reduction
methods, namely the TSM, the one-end trick ..., time-dilution and the Hopping Parameter Expansion (HPE) [7]".

With A = 1 + 2 i kappa mu g5 and H = A - M:  M^-1 = sum_{k<n} (A^-1 H)^k A^-1 + (A^-1 H)^n M^-1  for every n.
Everything below is checked against dense matrices assembled in tests/dense_ref.py (independent of the oracle) or
against closed forms worked out by hand from the hop structure.
"""
import numpy as np
import pytest

import dense_ref as dr
from paper_1401_6750_b200 import inputs
from test_oracle_operator import gauge_transform
from test_oracle_time_dilution import _dense_X


def dense_A(dims, kappa, mu):
    V = int(np.prod(dims))
    return np.eye(V * 12, dtype=complex) + 2j * kappa * mu * np.kron(np.eye(V), np.kron(dr.GAMMA5, np.eye(3)))


def projected_trace(Mat, X, dims, mom):
    """sum_{x in t} e^{ipx} tr_{spin,colour}[(X Mat)(x,x)] -> [nmom, T] from dense matrices."""
    lx, ly, lz, lt = dims
    V = int(np.prod(dims))
    diag = np.diag(X @ Mat)
    per_site = diag.reshape(V, 12).sum(1).reshape(lt, lz, ly, lx)
    xs = np.arange(lx)[None, None, :]
    ys = np.arange(ly)[None, :, None]
    zs = np.arange(lz)[:, None, None]
    out = np.empty((len(mom), lt), dtype=complex)
    for k, (px, py, pz) in enumerate(mom):
        ph = np.exp(2j * np.pi * (px * xs / lx + py * ys / ly + pz * zs / lz))
        out[k] = (per_site * ph[None]).sum(axis=(1, 2, 3))
    return out


@pytest.mark.parametrize("tb", [-1, 1])
def test_AinvH_vs_dense(orc, tb):
    """orc_apply_AinvH = A^-1 (A - M) with both factors assembled densely (catches a wrong sign of the twist in A^-1,
    H taken as M - A, a missing kappa)."""
    dims = (2, 2, 2, 4)
    k, mu = 0.15, 0.3
    U = inputs.gauge_field(dims, 0.3, 81)
    v = inputs.random_spinor(dims, 7)
    A = dense_A(dims, k, mu)
    M = dr.dense_M(U, dims, k, mu, tb)
    want = np.linalg.solve(A, (A - M) @ v.reshape(-1))
    got = orc.apply_AinvH(v, U, k, mu, tb).reshape(-1)
    assert np.allclose(got, want, atol=1e-13)
    # the factor is kappa D up to the site-local A^-1: linear in kappa at mu = 0
    g1 = orc.apply_AinvH(v, U, k, 0.0, tb)
    g2 = orc.apply_AinvH(v, U, 2 * k, 0.0, tb)
    assert np.allclose(g2, 2 * g1, atol=1e-13)


@pytest.mark.parametrize("order", [0, 1, 2, 3, 4])
def test_expansion_identity_and_exact_part_vs_dense(orc, order):
    """On 2^4 with a dense inverse, for all 80 insertions and several momenta:
       (i)  hpe_exact(n_loc, n_der) = projected trace of X_i sum_{k<n_i} (A^-1 H)^k A^-1 from dense matrices
       (ii) projected trace of X_i M^-1 = exact part + projected trace of X_i (A^-1 H)^{n_i} M^-1."""
    dims = (2, 2, 2, 2)
    tb = -1
    k, mu = 0.12, 0.25
    U = inputs.gauge_field(dims, 0.4, 83)
    mom = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 1]], dtype=np.int32)
    n_loc, n_der = orc.hpe_orders(order)
    assert (n_loc, n_der) == (order, min(order, 2))
    A = dense_A(dims, k, mu)
    M = dr.dense_M(U, dims, k, mu, tb)
    Ainv, Minv = np.linalg.inv(A), np.linalg.inv(M)
    AH = Ainv @ (A - M)
    X = _dense_X(U, dims, tb)
    got = orc.hpe_exact(U, k, mu, mom, tb, n_loc, n_der)
    for i in range(80):
        n = n_loc if i < 16 else n_der
        S = sum((np.linalg.matrix_power(AH, kk) @ Ainv for kk in range(n)), np.zeros_like(A))
        want = projected_trace(S, X[i], dims, mom)
        assert np.allclose(got[i], want, atol=1e-11), i
        full = projected_trace(Minv, X[i], dims, mom)
        rem = projected_trace(np.linalg.matrix_power(AH, n) @ Minv, X[i], dims, mom)
        assert np.allclose(full, want + rem, atol=1e-10), i


def test_full_dilution_of_loops_hpe_is_the_exact_trace(orc):
    """Estimator pin: with the 12 V unit vectors as sources and their exact solutions, the sum of the HPE loops'
    remainders + the exact part is the trace of X M^-1 (the estimator is unbiased term by term)."""
    dims = (2, 2, 2, 2)
    tb = 1
    k, mu = 0.12, 0.25
    V = int(np.prod(dims))
    U = inputs.gauge_field(dims, 0.4, 85)
    mom = np.array([[0, 0, 0], [1, 0, 1]], dtype=np.int32)
    M = dr.dense_M(U, dims, k, mu, tb)
    Minv = np.linalg.inv(M)
    X = _dense_X(U, dims, tb)
    shape = (dims[3], dims[2], dims[1], dims[0], 4, 3)
    exact = orc.hpe_exact(U, k, mu, mom, tb, 4, 2)
    zero = np.zeros_like(exact)
    tot = np.zeros_like(exact)
    for j in range(12 * V):
        e = np.zeros(12 * V, dtype=complex)
        e[j] = 1.0
        tot += orc.loops_hpe(e.reshape(shape), Minv[:, j].reshape(shape), U, k, mu, mom, tb, 4, exact=zero)
    tot += exact
    for i in range(80):
        want = projected_trace(Minv, X[i], dims, mom)
        assert np.allclose(tot[i], want, atol=1e-10), i
    # order 0 is the plain estimator
    eta = inputs.z4_source(dims, 3, 0)
    s = (Minv @ eta.reshape(-1)).reshape(shape)
    assert np.allclose(orc.loops_hpe(eta, s, U, k, mu, mom, tb, 0), orc.plain_loops_project(eta, s, U, mom, tb), atol=1e-12)


def closed_form_exact_part(dims, kappa, mu, order):
    """Closed forms of the exact part when every extent is >= 4 (no path of <= 3 hops closes around the torus), from the
    hop structure alone (numpy 4x4 algebra with the Kronecker-product gammas of dense_ref):
      ultra-local Gamma_n:  k = 0: 3 tr[G B];  k = 2: out and back, links cancel (tb^2 = 1):
                            3 kappa^2 sum_mu tr[G B ((1-g_mu) B (1+g_mu) + (1+g_mu) B (1-g_mu)) B];  k = 1, 3: nothing closes
      Gamma_n D_m:          k = 1: the derivative's hop and one hop back: 3 kappa tr[G B g_m B];  k = 0: D_m has no diagonal
    times the number of sites of a timeslice, at p = 0 only."""
    a = 2 * kappa * mu
    B = (np.eye(4) - 1j * a * dr.GAMMA5) / (1 + a * a)
    one = np.eye(4)
    n3 = dims[0] * dims[1] * dims[2]
    out = np.zeros(80, dtype=complex)
    n_loc, n_der = order, min(order, 2)
    for n in range(16):
        G = dr.big_gamma(n)
        if n_loc >= 1:
            out[n] += 3 * np.trace(G @ B)
        if n_loc >= 3:
            for m in range(4):
                g = dr.GAMMA[m]
                out[n] += 3 * kappa ** 2 * np.trace(G @ B @ ((one - g) @ B @ (one + g) + (one + g) @ B @ (one - g)) @ B)
        if n_der >= 2:
            for m in range(4):
                out[16 + 16 * m + n] += 3 * kappa * np.trace(G @ B @ dr.GAMMA[m] @ B)
    return n3 * out


@pytest.mark.parametrize("order", [1, 2, 3, 4])
@pytest.mark.parametrize("tb", [-1, 1])
def test_exact_part_closed_form_and_gauge_independence(orc, order, tb):
    """On 4^4 the brute-force exact part must equal the closed forms: a constant per timeslice at p = 0, zero at p != 0,
    the same for any gauge field (links cancel along out-and-back paths)."""
    dims = (4, 4, 4, 4)
    k, mu = 0.14, 0.2
    mom = np.array([[0, 0, 0], [1, 0, 0], [0, -1, 1]], dtype=np.int32)
    n_loc, n_der = orc.hpe_orders(order)
    want = closed_form_exact_part(dims, k, mu, order)
    U = inputs.gauge_field(dims, 0.4, 87)
    got = orc.hpe_exact(U, k, mu, mom, tb, n_loc, n_der)
    assert np.allclose(got[:, 0, :], want[:, None], atol=1e-10)
    assert np.abs(got[:, 1:, :]).max() <= 1e-10
    if order == 4 and tb == -1:
        Ufree = np.zeros_like(U)
        Ufree[..., :, :] = np.eye(3)
        assert np.allclose(orc.hpe_exact(Ufree, k, mu, mom, tb, n_loc, n_der), got, atol=1e-10)
        # the ultra-local closed forms are real multiples of tr[G], tr[G g5]: only the scalar and g5 insertions survive
        nz = [n for n in range(16) if abs(want[n]) > 1e-12]
        assert nz == [0, 15]


def test_remainder_is_gauge_invariant_and_order_reduces_variance(orc):
    """loops_hpe of a gauge-transformed (U, eta, s) is unchanged; and on a small ensemble of Z4 sources the spread of
    the HPE estimator of the scalar loop is below the plain estimator's (what the expansion is for)."""
    dims = (4, 4, 4, 4)
    tb = -1
    k, mu = 0.14, 0.2
    mom = np.array([[0, 0, 0]], dtype=np.int32)
    U = inputs.gauge_field(dims, 0.4, 89)
    exact = orc.hpe_exact(U, k, mu, mom, tb, 4, 2)
    plain, hpe = [], []
    for r in range(6):
        eta = inputs.z4_source(dims, 11, r)
        s, _, tr, st = orc.solve(eta, U, k, mu, 1e-11, tb)
        assert st == 0
        plain.append(orc.plain_loops_project(eta, s, U, mom, tb))
        hpe.append(orc.loops_hpe(eta, s, U, k, mu, mom, tb, 4, exact=exact))
        if r == 0:
            g = inputs.random_su3_field(dims, 5)
            eg, sg = (np.einsum("...ab,...sb->...sa", g, f) for f in (eta, s))
            assert np.allclose(orc.loops_hpe(eg, sg, gauge_transform(U, g), k, mu, mom, tb, 4, exact=exact), hpe[0], atol=1e-9)
    plain, hpe = np.array(plain), np.array(hpe)
    # same mean within the noise, smaller spread for the scalar (i = 0) and pseudoscalar (i = 15) insertions
    for i in (0, 15):
        sp, sh = plain[:, i, 0, :].std(axis=0).mean(), hpe[:, i, 0, :].std(axis=0).mean()
        assert sh < 0.7 * sp, (i, sp, sh)
        assert abs(plain[:, i, 0, :].mean() - hpe[:, i, 0, :].mean()) < 3 * (sp + sh)
