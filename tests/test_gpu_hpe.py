"""GPU parity: Hopping Parameter Expansion of the plain loop estimator (DESIGN.md
reading 23) vs the oracle.

Bars as for the other contractions and solves: loops of a given (eta, s) pair 1e-12 (fp64) / 1e-5
(fp32) per block, for every order; the estimator's HP per-source arrays end to end <= 100 rho_HP; its combiner against
the oracle combiner on the GPU's own per-source arrays 1e-12; N_LP = N_HP identity 1e-10.  The CUDA path adds the exact
part from closed forms; the oracle computes it by brute force over all 12 V unit vectors.
"""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 1e-5}
C1 = inputs.CONFIGS["c1"]
LP = dict(sloppy="f16", outer="f32", recon=12, rho=1e-2, max_iter=500, delta=0.1)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=2000, delta=0.1)


def check_blocks(got, ref, tol):
    for name, sl in (("local", slice(0, 16)), ("deriv", slice(16, 80))):
        e = rel_l2(got[sl], ref[sl])
        assert e <= tol, (name, e)


@pytest.mark.parametrize("acc", ["f64", "f32"])
@pytest.mark.parametrize("dims,tb,kappa,mu", [((4, 4, 4, 8), -1, 0.156, 0.01), ((6, 4, 4, 4), 1, 0.14, 0.3)])
def test_loop_hpe_project_all_orders(orc, acc, dims, tb, kappa, mu):
    """Any (eta, s) pair (the expansion identity does not need M s = eta), orders 0..4, 19 momenta, both time
    boundaries, a large twist (the exact part's gamma5 component); order 0 = the plain bilinears."""
    t = tm()
    U = inputs.gauge_field(dims, 0.25, 41)
    eta = inputs.z4_source(dims, 43, 0)
    s = inputs.random_spinor(dims, 45)
    mom = inputs.momentum_list(2)
    with t.TmContext(dims, tb) as ctx:
        ctx.tm_load_gauge(U)
        for order in range(5):
            n_loc, n_der = orc.hpe_orders(order)
            exact = orc.hpe_exact(U, kappa, mu, mom, tb, n_loc, n_der)
            ref = orc.loops_hpe(eta, s, U, kappa, mu, mom, tb, order, exact=exact)
            got = to_np(ctx.loop_hpe_project(eta, s, kappa, mu, mom, order, t.PREC[acc]))
            assert got.shape == ref.shape == (80, len(mom), dims[3])
            check_blocks(got, ref, TOL[acc])
            # the exact part alone: with s = 0 only the closed forms remain
            only = to_np(ctx.loop_hpe_project(eta, np.zeros_like(s), kappa, mu, mom, order, t.PREC[acc]))
            assert np.abs(only - exact).max() <= 1e-11 * max(1.0, np.abs(exact).max())
        plain = to_np(ctx.loop_plain_project_timeslice(eta, s, mom, -1, t.PREC[acc]))
        assert np.array_equal(to_np(ctx.loop_hpe_project(eta, s, kappa, mu, mom, 0, t.PREC[acc])), plain)
        with pytest.raises(t.TmError) as e:
            ctx.loop_hpe_project(eta, s, kappa, mu, mom, 5, t.PREC[acc])
        assert e.value.status == t.TM_EARG
        with pytest.raises(t.TmError):
            ctx.loop_hpe_project(eta, s, kappa, mu, mom, 2, t.TM_F16)


def test_hpe_refuses_short_extents():
    t = tm()
    dims = (4, 4, 2, 4)
    U = inputs.gauge_field(dims, 0.25, 41)
    eta = inputs.z4_source(dims, 43, 0)
    mom = inputs.momentum_list(0)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        with pytest.raises(t.TmError) as e:
            ctx.loop_hpe_project(eta, eta, 0.15, 0.01, mom, 2, t.TM_F64)
        assert e.value.status == t.TM_EDIM
        ctx.loop_hpe_project(eta, eta, 0.15, 0.01, mom, 0, t.TM_F64)      # order 0 needs no closed forms


def test_hpe_estimator_c1(orc):
    """tsm_estimate_hpe at c1, order 4: decomposition as for the other TSM loops, ragged groups
    (5 LP sources = a group of 4 + 1), packed noise, sharding, and the variance against the plain estimator."""
    t = tm()
    dims = C1["dims"]
    k, mu = C1["kappa"], C1["mu"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(2)
    n_lp, n_hp = 5, 3
    exact = orc.hpe_exact(U, k, mu, mom, -1, 4, 2)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, info = ctx.tsm_estimate_hpe(n_lp, n_hp, k, mu, mom, LP, HP, 4, t.TM_F32, t.TM_F64,
                                             seed=C1["src_seed"], per_source=True)
        out, ps = to_np(out), to_np(ps)
        assert info["worst_resid_lp"] <= LP["rho"] and info["worst_resid_hp"] <= HP["rho"]
        assert info["iters_lp"] > 0 and info["iters_hp"] > 0 and info["launches"] > 0
        assert rel_l2(out, orc.tsm_combine(ps[:n_lp], ps[n_lp:])) <= 1e-12
        plain_hp = []
        for r in range(n_hp):
            eta = inputs.z4_source(dims, C1["src_seed"], r)
            s, _, tr, st = orc.solve(eta, U, k, mu, 1e-12, -1)
            assert st == 0 and tr <= 1e-12
            ref = orc.loops_hpe(eta, s, U, k, mu, mom, -1, 4, exact=exact)
            assert rel_l2(ps[n_lp + r], ref) <= 100 * HP["rho"]
            assert rel_l2(ps[r], ref) <= 20 * LP["rho"]            # LP arrays are O(rho_LP) close
            plain_hp.append(orc.plain_loops_project(eta, s, U, mom, -1))
        # what the expansion is for: the scalar loop's spread over the HP sources is smaller than the plain estimator's
        sp = np.array(plain_hp)[:, 0, 0, :].std(axis=0).mean()
        sh = ps[n_lp:, 0, 0, :].std(axis=0).mean()
        assert sh < sp
        z4 = np.stack([inputs.pack_z4(inputs.z4_exponents(dims, C1["src_seed"], r)) for r in range(n_lp)])
        out2, _, _ = ctx.tsm_estimate_hpe(n_lp, n_hp, k, mu, mom, LP, HP, 4, t.TM_F32, t.TM_F64, z4=z4)
        assert np.array_equal(to_np(out2), out)
        ctx.tm_set_option(t.TM_OPT_GROUP, 1)
        out3, _, _ = ctx.tsm_estimate_hpe(n_lp, n_hp, k, mu, mom, LP, HP, 4, t.TM_F32, t.TM_F64, seed=C1["src_seed"])
        ctx.tm_set_option(t.TM_OPT_GROUP, 0)
        assert np.array_equal(to_np(out3), out)
        _, ps_b, _ = ctx.tsm_estimate_hpe(2, 0, k, mu, mom, LP, HP, 4, t.TM_F32, t.TM_F64, seed=C1["src_seed"],
                                          per_source=True, src_first=1, src_stride=2)
        assert np.array_equal(to_np(ps_b), ps[[1, 3]])
        # N_LP = N_HP with identical parameters: the LP terms cancel, TSM = plain HP mean within 1e-10 [B:ns]
        out4, ps4, _ = ctx.tsm_estimate_hpe(2, 2, k, mu, mom, HP, HP, 4, t.TM_F64, t.TM_F64, seed=C1["src_seed"],
                                            per_source=True)
        assert rel_l2(to_np(out4), to_np(ps4)[2:].mean(0)) <= 1e-10
        # order 2 of the estimator against the oracle as well (one contraction per source instead of two)
        _, ps2, _ = ctx.tsm_estimate_hpe(1, 1, k, mu, mom, LP, HP, 2, t.TM_F32, t.TM_F64, seed=C1["src_seed"], per_source=True)
        eta = inputs.z4_source(dims, C1["src_seed"], 0)
        s, _, _, _ = orc.solve(eta, U, k, mu, 1e-12, -1)
        assert rel_l2(to_np(ps2)[1], orc.loops_hpe(eta, s, U, k, mu, mom, -1, 2)) <= 100 * HP["rho"]
