"""GPU parity: time dilution (reading 22) vs the oracle.

Bars as for the other contractions and solves: plain bilinears of a given pair 1e-12 (fp64) / 1e-5
(fp32) per block; the estimator's HP per-noise-vector arrays end to end <= 100 rho_HP; its combiner against the oracle
combiner on the GPU's own per-noise-vector arrays 1e-12; N_LP = N_HP identity 1e-10.
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
@pytest.mark.parametrize("dims,p2,tb", [((4, 4, 4, 8), 4, -1), ((6, 4, 6, 10), 4, 1), ((8, 8, 8, 4), 9, -1)])
def test_plain_bilinears(orc, acc, dims, p2, tb):
    """loop_plain_project_timeslice on any pair (a, b): one timeslice (first, middle, last: the t-derivative reaches
    across the boundary) and the whole vector."""
    t = tm()
    U = inputs.gauge_field(dims, 0.25, 7)
    a = inputs.z4_source(dims, 207, 0)
    b = inputs.random_spinor(dims, 107)
    mom = inputs.momentum_list(p2)
    T = dims[3]
    ref = orc.plain_loops_project(a, b, U, mom, tb)
    with t.TmContext(dims, tb) as ctx:
        ctx.tm_load_gauge(U)
        got = to_np(ctx.loop_plain_project_timeslice(a, b, mom, -1, t.PREC[acc]))
        assert got.shape == ref.shape == (80, len(mom), T)
        check_blocks(got, ref, TOL[acc])
        for t0 in (0, T // 2, T - 1):
            one = to_np(ctx.loop_plain_project_timeslice(a, b, mom, t0, t.PREC[acc]))
            check_blocks(one[:, :, t0], ref[:, :, t0], TOL[acc])
            assert np.count_nonzero(np.delete(one, t0, axis=2)) == 0


def test_time_diluted_estimator_c1(orc):
    """tsm_estimate_time_diluted at c1 (4^3x8: 8 diluted sources per noise vector = one group of 8): decomposition as
    for the undiluted TSM loop."""
    t = tm()
    dims = C1["dims"]
    k, mu = C1["kappa"], C1["mu"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(2)
    n_lp, n_hp = 3, 2
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, info = ctx.tsm_estimate_time_diluted(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64,
                                                      seed=C1["src_seed"], per_source=True)
        out, ps = to_np(out), to_np(ps)
        assert info["worst_resid_lp"] <= LP["rho"] and info["worst_resid_hp"] <= HP["rho"]
        assert info["iters_lp"] > 0 and info["iters_hp"] > info["iters_lp"] and info["launches"] > 0
        # the combiner on the GPU's own per-noise-vector arrays
        assert rel_l2(out, orc.tsm_combine(ps[:n_lp], ps[n_lp:])) <= 1e-12
        # HP arrays end to end against the oracle's step-by-step time-diluted loops (unique solutions)
        for r in range(n_hp):
            eta = inputs.z4_source(dims, C1["src_seed"], r)
            ref, worst = orc.loops_time_diluted(eta, U, k, mu, 1e-12, mom, -1)
            assert worst <= 1e-12
            assert rel_l2(ps[n_lp + r], ref) <= 100 * HP["rho"]
            assert rel_l2(ps[r], ref) <= 20 * LP["rho"]            # LP arrays are O(rho_LP) close
        # packed noise from the host generator == device-generated noise; groups of 2 == groups of 8 (bit-identical)
        z4 = np.stack([inputs.pack_z4(inputs.z4_exponents(dims, C1["src_seed"], r)) for r in range(n_lp)])
        out2, _, _ = ctx.tsm_estimate_time_diluted(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, z4=z4)
        assert np.array_equal(to_np(out2), out)
        ctx.tm_set_option(t.TM_OPT_GROUP, 2)
        out3, _, _ = ctx.tsm_estimate_time_diluted(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=C1["src_seed"])
        ctx.tm_set_option(t.TM_OPT_GROUP, 0)
        assert np.array_equal(to_np(out3), out)
        # N_LP = N_HP with identical parameters: the LP terms cancel, TSM = plain HP mean within 1e-10 [B:ns]
        out4, ps4, _ = ctx.tsm_estimate_time_diluted(2, 2, k, mu, mom, HP, HP, t.TM_F64, t.TM_F64, seed=C1["src_seed"],
                                                     per_source=True)
        assert rel_l2(to_np(out4), to_np(ps4)[2:].mean(0)) <= 1e-10


def test_time_diluted_ragged_groups_and_sharding(orc):
    """T = 6 (one group of 4 + one of 2 diluted sources per noise vector), f64 contraction of an f32-outer LP pass
    (precision conversion + re-expanded noise), and source sharding: the arrays of global sources 1, 3 from a call
    with src_first = 1, src_stride = 2 equal those of a 4-source run."""
    t = tm()
    dims = (4, 4, 4, 6)
    k, mu = 0.156, 0.01
    U = inputs.gauge_field(dims, 0.3, 11)
    mom = inputs.momentum_list(1)
    lp = dict(LP, sloppy="bf16")
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        _, ps, _ = ctx.tsm_estimate_time_diluted(4, 1, k, mu, mom, lp, HP, t.TM_F64, t.TM_F64, seed=21, per_source=True)
        ps = to_np(ps)
        eta = inputs.z4_source(dims, 21, 0)
        ref, _ = orc.loops_time_diluted(eta, U, k, mu, 1e-12, mom, -1)
        assert rel_l2(ps[4], ref) <= 100 * HP["rho"]
        assert rel_l2(ps[0], ref) <= 20 * lp["rho"]
        _, ps_b, _ = ctx.tsm_estimate_time_diluted(2, 0, k, mu, mom, lp, HP, t.TM_F64, t.TM_F64, seed=21, per_source=True,
                                                   src_first=1, src_stride=2)
        assert np.array_equal(to_np(ps_b), ps[[1, 3]])
