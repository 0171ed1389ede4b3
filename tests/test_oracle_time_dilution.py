"""Pins for the oracle's time-dilution functions (reading 22).

PAPER.md:88 "we also worked with time-dilution [6], so there are GPU kernels to contract a single time slice or a
whole vector"; PAPER.md:92 lists time-dilution among the variance-reduction methods of the code.
"""
import numpy as np

import dense_ref as dr
from paper_1401_6750_b200 import inputs
from test_oracle_operator import gauge_transform


def _dense_X(U, dims, tb):
    """The 80 insertions X_i as dense (12V x 12V) matrices from dense_ref (independent of the oracle)."""
    V = int(np.prod(dims))
    Dm = [dr.dense_cov_deriv(U, dims, m, tb) for m in range(4)]
    X = []
    for n in range(16):
        X.append(np.kron(np.eye(V), np.kron(dr.big_gamma(n), np.eye(3))))
    for m in range(4):
        for n in range(16):
            X.append(X[n] @ Dm[m])
    return X


def test_time_dilute_is_a_mask(orc):
    dims = (4, 2, 2, 4)
    eta = inputs.z4_source(dims, 5, 0)
    tot = np.zeros_like(eta)
    for t0 in range(dims[3]):
        e = orc.time_dilute(eta, t0)
        assert np.array_equal(e[t0], eta[t0])
        assert np.count_nonzero(e) == np.count_nonzero(eta[t0])
        tot += e
    assert np.array_equal(tot, eta)             # the diluted sources partition the noise vector


def test_plain_bilinears_vs_dense_einsum(orc):
    """orc_plain_loops_project against a^dag X_i b written out with numpy and the dense D_m, per timeslice, for a
    momentum list with unequal extents (catches a transposed operand, a gamma5 left in, a wrong derivative side)."""
    dims = (4, 2, 2, 4)
    tb = -1
    lx, ly, lz, lt = dims
    V = int(np.prod(dims))
    U = inputs.gauge_field(dims, 0.3, 71)
    a = inputs.random_spinor(dims, 3)
    b = inputs.random_spinor(dims, 4)
    mom = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [-1, 1, 1], [2, 0, -1]], dtype=np.int32)
    got = orc.plain_loops_project(a, b, U, mom, tb)
    X = _dense_X(U, dims, tb)
    av, bv = a.reshape(-1), b.reshape(-1)
    xs = np.arange(lx)[None, None, :]
    ys = np.arange(ly)[None, :, None]
    zs = np.arange(lz)[:, None, None]
    for i in (0, 1, 5, 10, 15, 16, 16 + 7, 32 + 2, 48 + 9, 64 + 15):
        per_site = (av.conj() * (X[i] @ bv)).reshape(V, 12).sum(1).reshape(lt, lz, ly, lx)
        for k, (px, py, pz) in enumerate(mom):
            ph = np.exp(2j * np.pi * (px * xs / lx + py * ys / ly + pz * zs / lz))
            want = (per_site * ph[None]).sum(axis=(1, 2, 3))
            assert np.allclose(got[i, k], want, atol=1e-11), (i, k)
    # restricted timeslice window leaves the other columns zero
    one = orc.plain_loops_project(a, b, U, mom, tb, 2, 3)
    assert np.array_equal(one[:, :, 2], got[:, :, 2]) and np.count_nonzero(np.delete(one, 2, axis=2)) == 0


def test_exact_dilution_of_one_timeslice_vs_dense_trace(orc):
    """Reading 22 pinned exactly on 2^4: replace the noise on timeslice t0 by all 12 V3 unit vectors e_r of that
    timeslice (exact spin-colour-site dilution).  Then
        sum_r  e_r^dag X_i s_r  (contracted on timeslice t0)  =  sum_{x in t0} tr[X_i M^-1](x,x)
    with s_r = M^-1 e_r from numpy LU: the plain time-diluted estimator is unbiased for the loop on its timeslice."""
    dims = (2, 2, 2, 2)
    V, V3 = 16, 8
    k, mu, tb = 0.156, 0.05, -1
    U = inputs.gauge_field(dims, 0.3, 61)
    S = np.linalg.inv(dr.dense_M(U, dims, k, mu, tb))
    X = _dense_X(U, dims, tb)
    mom = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 1]], dtype=np.int32)
    for t0 in range(2):
        acc = np.zeros((80, len(mom)), dtype=complex)
        for r in range(t0 * V3 * 12, (t0 + 1) * V3 * 12):
            e = np.zeros(12 * V, dtype=complex)
            e[r] = 1
            shape = (2, 2, 2, 2, 4, 3)
            ed = orc.time_dilute(e.reshape(shape), t0)
            assert np.array_equal(ed.reshape(-1), e)
            acc += orc.plain_loops_project(ed, S[:, r].copy().reshape(shape), U, mom, tb, t0, t0 + 1)[:, :, t0]
        for i in range(80):
            A = X[i] @ S
            d = np.array([np.trace(A[x * 12:(x + 1) * 12, x * 12:(x + 1) * 12]) for x in range(t0 * V3, (t0 + 1) * V3)])
            d = d.reshape(2, 2, 2)                  # [z][y][x] of timeslice t0
            for q, (px, py, pz) in enumerate(mom):
                zz, yy, xx = np.meshgrid(np.arange(2), np.arange(2), np.arange(2), indexing="ij")
                want = (d * np.exp(2j * np.pi * (px * xx / 2 + py * yy / 2 + pz * zz / 2))).sum()
                assert abs(acc[i, q] - want) <= 1e-10, (t0, i, q)


def test_time_diluted_loops_linearity_and_gauge_invariance(orc):
    """loops_time_diluted (solve per timeslice + single-timeslice contraction): (a) its column t0 is the diagonal
    block of B[t, t0] = eta^(t)^dag X s^(t0); summing the blocks over t0 gives the undiluted bilinear eta^dag X s with
    s = sum_t0 s^(t0) = M^-1 eta (linearity of the solve); (b) invariant under a gauge transformation."""
    dims = (4, 2, 2, 4)
    k, mu, tb = 0.15, 0.05, -1
    T = dims[3]
    U = inputs.gauge_field(dims, 0.3, 71)
    eta = inputs.z4_source(dims, 72, 0)
    mom = np.array([[0, 0, 0], [1, 0, 0], [0, -1, 1]], dtype=np.int32)
    got, worst = orc.loops_time_diluted(eta, U, k, mu, 1e-12, mom, tb)
    assert worst <= 1e-12
    s_full, _, _, st = orc.solve(eta, U, k, mu, 1e-13, tb)
    assert st == 0
    undiluted = orc.plain_loops_project(eta, s_full, U, mom, tb)
    blocks = np.zeros_like(undiluted)
    for t0 in range(T):
        s_t0, _, _, st = orc.solve(orc.time_dilute(eta, t0), U, k, mu, 1e-13, tb)
        assert st == 0
        full = orc.plain_loops_project(eta, s_t0, U, mom, tb)       # B[t, t0] for every t
        assert np.allclose(full[:, :, t0], got[:, :, t0], atol=1e-9)
        blocks += full
    assert np.allclose(blocks, undiluted, atol=1e-8)
    assert not np.allclose(got, undiluted, atol=1e-3)               # the cross terms are really dropped
    # gauge invariance of the time-diluted loops
    g = inputs.random_su3_field(dims, 9)
    Ug, etag = gauge_transform(U, g), np.einsum("...ab,...sb->...sa", g, eta)
    got_g, _ = orc.loops_time_diluted(etag, Ug, k, mu, 1e-12, mom, tb)
    assert np.allclose(got_g, got, atol=1e-9)


def test_plain_loops_from_the_generalised_one_end_primitive(orc):
    """The identity the CUDA path uses to get the plain bilinears out of its 160-insertion primitive (DESIGN.md
    reading 22): with mu = 0 the primitive's f = 1 block of the swapped pair is a^dag g5 G_n D g5 b, and
    g5 G_n g5 = eps_n G_n, so  a^dag G_n D b = eps_n * loops_project(s := a, eta := b, mu = 0)[1]."""
    dims = (4, 2, 2, 4)
    tb = -1
    U = inputs.gauge_field(dims, 0.3, 71)
    a = inputs.random_spinor(dims, 3)
    b = inputs.random_spinor(dims, 4)
    mom = np.array([[0, 0, 0], [1, 0, 0], [0, 1, -1]], dtype=np.int32)
    plain = orc.plain_loops_project(a, b, U, mom, tb)
    prim = orc.loops_project(a, b, U, 0.123, 0.0, mom, tb)[1]
    g5 = dr.GAMMA5
    for i in range(80):
        n = i if i < 16 else (i - 16) & 15
        G = dr.big_gamma(n)
        W = g5 @ G @ g5
        eps = 1.0 if np.allclose(W, G) else -1.0
        assert np.allclose(W, eps * G)
        assert np.allclose(plain[i], eps * prim[i], atol=1e-11), i
