"""Pins for the oracle's 160 insertions, momentum projection and TSM combiner.

PAPER.md:72 (one-end trick, 160 insertions, p^2 <= 9), :86 (colour trace, open Dirac indices,
covariant derivative), :88/:94-100 (time-slice-indexed output, Fourier transform), :58 (TSM).
"""
import os

import numpy as np
import pytest

import dense_ref as dr
from paper_1401_6750_b200 import inputs
from test_oracle_operator import gauge_transform


def test_momentum_counts():
    """PAPER.md:72 'up to p^2 <= 9': 123 integer vectors; 33 for p^2 <= 4 (BASELINE c3); 1 for p = 0."""
    assert len(inputs.momentum_list(9)) == 123
    assert len(inputs.momentum_list(4)) == 33
    assert len(inputs.momentum_list(0)) == 1
    m = inputs.momentum_list(9)
    assert tuple(m[0]) == (0, 0, 0)
    assert len({tuple(r) for r in m}) == 123
    assert {tuple(r) for r in m} == {tuple(-r) for r in m}
    assert np.all(np.diff((m.astype(int) ** 2).sum(1)) >= 0)


def test_full_dilution_vs_dense_traces(orc):
    """Exact check of the one-end-trick reading (readings 4,5) on 2^4: replacing the
    noise by all 12V unit vectors e_r (s_r = column r of M_u^-1, from numpy LU),
      sum_r l_r[0][i](x) = Tr_x[X (M_u^-1 - M_d^-1)] / (-4 i kappa mu)
      sum_r l_r[1][i](x) = Tr_x[X (M_u^-1 + M_d^-1)] / 2
    with X = Gamma_n (i = n) or Gamma_n D_m (i = 16+16m+n), Tr_x over spin-colour at site x."""
    dims = (2, 2, 2, 2)
    V = 16
    k, mu, tb = 0.156, 0.05, -1
    U = inputs.gauge_field(dims, 0.3, 61)
    Mu = dr.dense_M(U, dims, k, mu, tb)
    Md = dr.dense_M(U, dims, k, -mu, tb)
    Su, Sd = np.linalg.inv(Mu), np.linalg.inv(Md)
    acc = np.zeros((V, 2, 80), dtype=complex)
    for r in range(12 * V):
        e = np.zeros(12 * V, dtype=complex)
        e[r] = 1
        s = Su[:, r].copy().reshape(2, 2, 2, 2, 4, 3)
        acc += orc.loops_sites(s, e.reshape(s.shape), U, k, mu, tb=tb)
    diff_ud = (Su - Sd) / (-4j * k * mu)
    sum_ud = (Su + Sd) / 2
    Dm = [dr.dense_cov_deriv(U, dims, m, tb) for m in range(4)]
    for n in range(16):
        Gn = np.kron(np.eye(V), np.kron(dr.big_gamma(n), np.eye(3)))
        for blk, X in [(n, Gn)] + [(16 + 16 * m + n, Gn @ Dm[m]) for m in range(4)]:
            for f, P in [(0, diff_ud), (1, sum_ud)]:
                A = X @ P
                want = np.array([np.trace(A[x * 12:(x + 1) * 12, x * 12:(x + 1) * 12]) for x in range(V)])
                assert np.allclose(acc[:, f, blk], want, atol=1e-10), (n, blk, f)


@pytest.fixture(scope="module")
def small_case(orc):
    dims = (4, 2, 2, 4)
    k, mu, tb = 0.156, 0.03, -1
    U = inputs.gauge_field(dims, 0.3, 71)
    eta = inputs.z4_source(dims, 72, 0)
    s, _, _, _ = orc.solve(eta, U, k, mu, 1e-2)     # deliberately inexact: M s != eta
    return dims, k, mu, tb, U, eta, s


def test_loops_explicit_bilinears(orc, small_case):
    """l[f][i](x) against numpy einsum with dense_ref gammas and the oracle-independent dense D_m."""
    dims, k, mu, tb, U, eta, s = small_case
    V = int(np.prod(dims))
    l = orc.loops_sites(s, eta, U, k, mu, tb=tb)
    sf = s.reshape(V, 4, 3)
    g = np.einsum("ab,xbc->xac", dr.GAMMA5, eta.reshape(V, 4, 3)) - 2j * k * mu * sf
    fam = [sf, g]
    for f in range(2):
        for n in range(16):
            X = dr.GAMMA5 @ dr.big_gamma(n)
            want = np.einsum("xac,ab,xbc->x", sf.conj(), X, fam[f])
            assert np.allclose(l[:, f, n], want, atol=1e-12)
            for m in range(4):
                d = (dr.dense_cov_deriv(U, dims, m, tb) @ fam[f].ravel()).reshape(V, 4, 3)
                want = np.einsum("xac,ab,xbc->x", sf.conj(), X, d)
                assert np.allclose(l[:, f, 16 + 16 * m + n], want, atol=1e-12)


def test_loops_norm_and_reality(orc, small_case):
    dims, k, mu, tb, U, eta, s = small_case
    l = orc.loops_sites(s, eta, U, k, mu, tb=tb)
    # g5 Gamma_15 = 1  =>  sum_x l[0][15] = ||s||^2
    assert abs(l[:, 0, 15].sum() - np.vdot(s, s)) < 1e-11 * abs(np.vdot(s, s))
    # s^dag H s is real wherever g5 Gamma_n is Hermitian
    herm = [n for n in range(16)
            if np.allclose(dr.GAMMA5 @ dr.big_gamma(n), (dr.GAMMA5 @ dr.big_gamma(n)).conj().T)]
    assert herm == [0, 7, 11, 13, 14, 15]
    for n in range(16):
        im = np.abs(l[:, 0, n].imag).max()
        re = np.abs(l[:, 0, n].real).max()
        if n in herm:
            assert im < 1e-12
        else:
            assert re < 1e-12     # anti-Hermitian -> purely imaginary
    # reading 5: with an exact solve, g = g5 D_W s; here check the residual identity
    # g(from eta) - g5 D_W s = g5 (eta - M s),  D_W = M - 2 i kappa mu g5
    g5 = np.array([1, 1, -1, -1]).reshape(4, 1)
    Ms = orc.apply_M(s, U, k, mu, tb)
    DWs = Ms - 2j * k * mu * g5 * s
    g = g5 * eta - 2j * k * mu * s
    assert np.allclose(g - g5 * DWs, g5 * (eta - Ms), atol=1e-13)


def test_loops_gauge_invariance(orc, small_case):
    """all 160 insertions invariant under (U, s, eta) -> (U^g, g s, g eta)  [B:ns]."""
    dims, k, mu, tb, U, eta, s = small_case
    g = inputs.random_su3_field(dims, 73)
    rot = lambda v: np.einsum("...ab,...sb->...sa", g, v)
    a = orc.loops_sites(s, eta, U, k, mu, tb=tb)
    b = orc.loops_sites(rot(s), rot(eta), gauge_transform(U, g), k, mu, tb=tb)
    assert np.abs(a - b).max() < 1e-12 * np.abs(a).max()


def test_summation_by_parts(orc, small_case):
    """sum_x s^dag X D_m psi = - sum_x (D_m s)^dag X psi (D_m anti-Hermitian, X site-independent)."""
    dims, k, mu, tb, U, eta, s = small_case
    V = int(np.prod(dims))
    l = orc.loops_sites(s, eta, U, k, mu, tb=tb).sum(axis=0)
    for m in range(4):
        ds = orc.cov_deriv(s, U, m, tb).reshape(V, 4, 3)
        for n in (0, 3, 9, 15):
            X = dr.GAMMA5 @ dr.big_gamma(n)
            want = -np.einsum("xac,ab,xbc->", ds.conj(), X, s.reshape(V, 4, 3))
            assert abs(l[0, 16 + 16 * m + n] - want) < 1e-11 * max(1, abs(want))


def test_project_vs_numpy_fft(orc, small_case):
    """out[f,i,k,t] = L^3 * ifftn(l[t], axes=(z,y,x))[pz,py,px]  (+i convention, reading 15);
    p = 0 is the plain timeslice sum."""
    dims, k, mu, tb, U, eta, s = small_case
    lx, ly, lz, lt = dims
    mom = inputs.momentum_list(9)
    out = orc.loops_project(s, eta, U, k, mu, mom, tb=tb)
    assert out.shape == (2, 80, 123, lt)
    l = orc.loops_sites(s, eta, U, k, mu, tb=tb).reshape(lt, lz, ly, lx, 2, 80)
    ft = np.fft.ifftn(l, axes=(1, 2, 3)) * (lx * ly * lz)
    for q, (px, py, pz) in enumerate(mom):
        want = ft[:, pz % lz, py % ly, px % lx]          # [t, 2, 80]
        assert np.allclose(out[:, :, q, :], np.moveaxis(want, 0, -1), atol=1e-11)
    assert np.allclose(out[:, :, 0, :], np.moveaxis(l.sum(axis=(1, 2, 3)), 0, -1), atol=1e-11)
    # timeslice window leaves the rest untouched (zero)
    part = orc.loops_project(s, eta, U, k, mu, mom[:5], tb=tb, t0=1, t1=3)
    assert np.allclose(part[..., 1:3], out[:, :, :5, 1:3]) and np.all(part[..., 0] == 0) and np.all(part[..., 3] == 0)


def test_project_delta(orc):
    """asymmetric extents: a loop field ~ e^{-2 pi i q.x/L} projects to L^3 delta_{pq}.
    Built from s = eta-independent trick: s = plane wave in colour/spin component 0 only, U = 1,
    l[0][15] = |s|^2 is constant -> only p = 0 survives with value V3 * |u|^2."""
    dims = (4, 6, 2, 2)
    lx, ly, lz, lt = dims
    t, z, y, x = np.meshgrid(np.arange(lt), np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    q = (1, -2, 1)
    s = np.zeros((lt, lz, ly, lx, 4, 3), dtype=complex)
    s[..., 0, 0] = 1.0
    eta = np.zeros_like(s)
    # eta = g5-component carrying the phase so that l[1][0] = s^dag g5 g = s^dag eta-part = e^{-iqx}
    eta[..., 0, 0] = np.exp(-2j * np.pi * (q[0] * x / lx + q[1] * y / ly + q[2] * z / lz))
    mom = np.array([[0, 0, 0], list(q), [-q[0], -q[1], -q[2]], [1, 0, 0]], dtype=np.int32)
    out = orc.loops_project(s, eta, inputs.unit_gauge(dims), 0.1, 0.0, mom, tb=1)
    V3 = lx * ly * lz
    # f=1, n=0: s^dag g5 (g5 eta) = conj(s00) eta00 = e^{-iqx}
    assert np.allclose(out[1, 0, :, :], np.array([0, V3, 0, 0])[:, None], atol=1e-10)
    assert np.allclose(out[0, 15, :, :], np.array([V3, 0, 0, 0])[:, None], atol=1e-10)


def test_tsm_combine(orc):
    """PAPER.md:58 + reading 14.  Hand-computed example and the N_LP = N_HP identity [B:ns]."""
    lp = np.array([[1 + 1j, 2], [3, 4], [5, 6 - 2j], [7, 8]], dtype=complex)
    hp = np.array([[1.5 + 1j, 2.5], [2, 4.25]], dtype=complex)
    got = orc.tsm_combine(lp, hp)
    # mean(lp) = [4+0.25j, 5-0.5j]; correction = mean(hp - lp[:2]) = [(0.5 - 1)/2, (0.5 + 0.25)/2]
    assert np.allclose(got, [4 + 0.25j - 0.25, 5 - 0.5j + 0.375])
    golden = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "tsm_example.txt"))
    assert np.allclose(got, golden[:, 0] + 1j * golden[:, 1])
    rng = np.random.default_rng(3)
    lp = rng.normal(size=(5, 7)) + 1j * rng.normal(size=(5, 7))
    hp = rng.normal(size=(5, 7)) + 1j * rng.normal(size=(5, 7))
    assert np.allclose(orc.tsm_combine(lp, hp), hp.mean(axis=0), atol=1e-14)   # N_LP = N_HP
    assert np.allclose(orc.tsm_combine(lp, hp[:0]), lp.mean(axis=0), atol=1e-14)  # no correction
    hp3 = hp[:3]
    assert np.allclose(orc.tsm_combine(lp, hp3), lp.mean(0) + (hp3 - lp[:3]).mean(0), atol=1e-14)


def test_binary_storage_fig2(orc):
    """sec 2.1.1 / Fig. 2: the 13-source example, hand-worked in tests/golden/binary_storage_example.txt."""
    v = (np.arange(15) + 1.0).astype(np.complex128).reshape(15, 1)
    files, counts = orc.binary_store(v)
    assert list(counts) == [1, 2, 4, 8]
    assert np.allclose(files[:, 0], [1, 5, 22, 92])
    golden = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "binary_storage_example.txt"))
    for N, tot in golden:
        got = orc.binary_recover(files, counts, int(N))
        assert got is not None and abs(got[0] - tot / N) < 1e-14, (N, got)
    # 13 = 1101b uses exactly the sources {0} + {3..6} + {7..14}: brute force over those subsets
    rng = np.random.default_rng(3)
    ps = rng.normal(size=(15, 4, 3)) + 1j * rng.normal(size=(15, 4, 3))
    files, counts = orc.binary_store(ps)
    sel = [0] + list(range(3, 7)) + list(range(7, 15))
    assert len(sel) == 13
    assert np.allclose(orc.binary_recover(files, counts, 13), ps[sel].mean(axis=0), atol=1e-14)
    # any N <= 15 is recoverable and is a mean over N distinct sources; a full set is the plain mean
    for N in range(1, 16):
        sel = [r for k in range(4) if (N >> k) & 1 for r in range(2 ** k - 1, 2 ** (k + 1) - 1)]
        assert len(sel) == N
        assert np.allclose(orc.binary_recover(files, counts, N), ps[sel].mean(axis=0), atol=1e-14)
    assert np.allclose(orc.binary_recover(files, counts, 15), ps.mean(axis=0), atol=1e-14)
    # an incomplete last file (13 sources generated) cannot serve N = 8..12, 14, 15; the complete ones still serve
    # N <= 7, and N = 13 = everything stored so far is the sum of every file, the partial one included
    # ("one can recover the data for any number of sources"): nothing is lost
    files, counts = orc.binary_store(ps[:13])
    assert list(counts) == [1, 2, 4, 6]
    for N in (8, 9, 12, 14, 15, 16):
        assert orc.binary_recover(files, counts, N) is None
    assert np.allclose(orc.binary_recover(files, counts, 7), ps[:7].mean(axis=0), atol=1e-14)
    assert np.allclose(orc.binary_recover(files, counts, 13), ps[:13].mean(axis=0), atol=1e-14)
    # the headline run: 500 LP sources and 20 corrections are recoverable in full, brute force on the plain means
    for n in (500, 20):
        big = rng.normal(size=(n, 3)) + 1j * rng.normal(size=(n, 3))
        files, counts = orc.binary_store(big)
        assert int(counts.sum()) == n and counts[-1] != 2 ** (len(counts) - 1)
        assert np.allclose(orc.binary_recover(files, counts, n), big.mean(axis=0), atol=1e-13)
        full = 2 ** (len(counts) - 1) - 1                # the largest complete prefix (255 | 15)
        assert np.allclose(orc.binary_recover(files, counts, full), big[:full].mean(axis=0), atol=1e-13)
    # O(log2 N) files
    assert [orc.binary_nfiles(n) for n in (1, 2, 3, 4, 7, 8, 500, 1023)] == [1, 2, 2, 3, 3, 4, 9, 10]


def test_explicit_dw_variant(orc):
    """Row f3 / reading 5: with D_W applied explicitly the f = 1 loops differ from the eta-based ones by the
    bilinears of gamma5 (eta - M s); they coincide when M s = eta."""
    dims = (4, 2, 2, 4)
    k, mu = 0.156, 0.01
    U = inputs.gauge_field(dims, 0.3, 11)
    s = inputs.random_spinor(dims, 12)
    eta = inputs.random_spinor(dims, 13)
    mom = inputs.momentum_list(1)
    a = orc.loops_project(s, eta, U, k, mu, mom, -1)
    b = orc.loops_project_explicit(s, U, k, mu, mom, -1)
    assert np.allclose(a[0], b[0], atol=1e-13)                      # f = 0 does not see eta
    # ultra-local f = 1 difference = sum_x e^{ipx} s^dag g5 Gamma_n g5 (eta - M s), written out with numpy
    r = eta - orc.apply_M(s, U, k, mu, -1)
    g5 = orc.gamma(4)
    lx, ly, lz, lt = dims
    for n in (0, 3, 9, 15):
        X = g5 @ orc.Gamma(n) @ g5
        site = np.einsum("tzyxac,ab,tzyxbc->tzyx", s.conj(), X, r)
        for kk, (px, py, pz) in enumerate(mom):
            ph = np.exp(2j * np.pi * (px * np.arange(lx)[None, None, :] / lx + py * np.arange(ly)[None, :, None] / ly
                                      + pz * np.arange(lz)[:, None, None] / lz))
            ref = (site * ph[None]).sum(axis=(1, 2, 3))
            assert np.allclose(a[1, n, kk] - b[1, n, kk], ref, atol=1e-12), (n, kk)
    # a true solution: both variants agree
    eta = inputs.z4_source(dims, 5, 0)
    s_sol, _, tr, st = orc.solve(eta, U, k, mu, 1e-13)
    assert st == 0
    a = orc.loops_project(s_sol, eta, U, k, mu, mom, -1)
    b = orc.loops_project_explicit(s_sol, U, k, mu, mom, -1)
    assert np.linalg.norm(a - b) <= 1e-10 * np.linalg.norm(a)


def test_symmetrised_derivative_explicit_bilinears(orc, small_case):
    """orc_loops_project_sym from its definition, written out with numpy and the oracle-independent dense D_m
    (dense_ref.dense_cov_deriv) acting on BOTH s and psi: for every timeslice, momentum, family f, direction m and all
    16 Gamma_n,   l_sym = sum_x e^{+ip.x} 1/2 [ s^dag g5 G_n (D_m psi) - (D_m s)^dag g5 G_n psi ](x),  psi = s | g.
    A wrong sign of the second term, a missing 1/2, a conjugation slip or a family mix-up fails this."""
    dims, k, mu, tb, U, eta, s = small_case
    lx, ly, lz, lt = dims
    V = int(np.prod(dims))
    mom = inputs.momentum_list(2)
    got = orc.loops_project_sym(s, eta, U, k, mu, mom, tb)
    sf = s.reshape(V, 4, 3)
    g = np.einsum("ab,xbc->xac", dr.GAMMA5, eta.reshape(V, 4, 3)) - 2j * k * mu * sf
    fam = [sf, g]
    zz, yy, xx = np.meshgrid(np.arange(lz), np.arange(ly), np.arange(lx), indexing="ij")
    phases = [np.exp(2j * np.pi * (px * xx / lx + py * yy / ly + pz * zz / lz)) for px, py, pz in mom]
    for m in range(4):
        D = dr.dense_cov_deriv(U, dims, m, tb)
        Ds = (D @ sf.ravel()).reshape(V, 4, 3)
        for f in range(2):
            Dpsi = (D @ fam[f].ravel()).reshape(V, 4, 3)
            for n in range(16):
                X = dr.GAMMA5 @ dr.big_gamma(n)
                site = 0.5 * (np.einsum("xac,ab,xbc->x", sf.conj(), X, Dpsi)
                              - np.einsum("xac,ab,xbc->x", Ds.conj(), X, fam[f]))
                site = site.reshape(lt, lz, ly, lx)
                for kk, ph in enumerate(phases):
                    want = (site * ph[None]).sum(axis=(1, 2, 3))
                    assert np.allclose(got[f, 16 + 16 * m + n, kk], want, atol=1e-12), (m, f, n, kk)
    # the ultra-local entries are the plain ones
    assert np.allclose(got[:, :16], orc.loops_project(s, eta, U, k, mu, mom, tb)[:, :16], atol=1e-13)


def test_symmetrised_derivative_variant(orc):
    """Row f3 / reading 4: D<-> = (D-> - D<-)/2.  Pins: summation by parts (D_mu is anti-Hermitian, so at p = 0 the
    symmetrised and the right-acting loops coincide); for f = 0 and Hermitian g5 Gamma_n the symmetrised insertion
    is i Im of the right-acting one at every site, hence its p = 0 projection is purely imaginary; gauge invariance."""
    dims = (4, 2, 2, 4)
    k, mu = 0.156, 0.01
    U = inputs.gauge_field(dims, 0.3, 21)
    s = inputs.random_spinor(dims, 22)
    eta = inputs.random_spinor(dims, 23)
    mom = inputs.momentum_list(1)
    a = orc.loops_project(s, eta, U, k, mu, mom, -1)
    b = orc.loops_project_sym(s, eta, U, k, mu, mom, -1)
    assert np.allclose(a[:, :16], b[:, :16], atol=1e-13)                      # ultra-local entries untouched
    # p = 0 (first momentum of the list), summed over t: D anti-Hermitian => sum_x (D s)^dag X psi = - sum_x s^dag X D psi
    assert tuple(mom[0]) == (0, 0, 0)
    assert np.allclose(a[:, 16:, 0].sum(axis=-1), b[:, 16:, 0].sum(axis=-1), atol=1e-11)
    assert np.abs(a[:, 16:] - b[:, 16:]).max() > 1e-3                          # but they differ mode by mode
    # f = 0, Hermitian g5 Gamma_n (n in {0, 7, 11, 13, 14, 15}): l_sym(x) = i Im l(x); at p = 0 per timeslice: purely imaginary
    for n in (0, 7, 11, 13, 14, 15):
        M = orc.gamma(4) @ orc.Gamma(n)
        assert np.allclose(M, M.conj().T)
        for m in range(4):
            i = 16 + 16 * m + n
            assert np.allclose(b[0, i, 0].real, 0, atol=1e-11)
            assert np.allclose(b[0, i, 0].imag, a[0, i, 0].imag, atol=1e-11)
    # gauge invariance under a random g(x) applied to (U, s, eta)
    rng = np.random.default_rng(5)
    lt, lz, ly, lx = s.shape[:4]
    h = rng.normal(size=(lt, lz, ly, lx, 3, 3)) + 1j * rng.normal(size=(lt, lz, ly, lx, 3, 3))
    q, _ = np.linalg.qr(h)
    q = q / np.linalg.det(q)[..., None, None] ** (1 / 3)
    Ug = np.empty_like(U)
    shifts = [(3, -1), (2, -1), (1, -1), (0, -1)]                              # x+mu for mu = x, y, z, t
    for m in range(4):
        ax, sh = shifts[m]
        Ug[..., m, :, :] = q @ U[..., m, :, :] @ np.roll(q, sh, axis=ax).conj().swapaxes(-1, -2)
    sg = np.einsum("...ab,...sb->...sa", q, s)
    eg = np.einsum("...ab,...sb->...sa", q, eta)
    # antiperiodic time boundary is a property of the fields, not of g(x): g is periodic, so the loops are invariant
    c = orc.loops_project_sym(sg, eg, Ug, k, mu, mom, -1)
    assert np.linalg.norm(c - b) <= 1e-11 * np.linalg.norm(b)
