"""GPU parity: the TSM estimator loop through the C ABI.

LP solutions are not unique, so the end-to-end check is by decomposition:
per-source arrays vs the oracle, the oracle's combiner on the GPU's per-source arrays, the
N_LP = N_HP identity (BASELINE.json north_star: within 1e-10), and path equivalences.
"""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
C1 = inputs.CONFIGS["c1"]
LP = dict(sloppy="bf16", outer="f32", recon=12, rho=1e-2, max_iter=500, delta=0.1)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=2000, delta=0.1)


def packed_z4(dims, seed, n):
    return np.stack([inputs.pack_z4(inputs.z4_exponents(dims, seed, r)) for r in range(n)])


@pytest.fixture(scope="module")
def setup():
    dims = C1["dims"]
    return dims, inputs.gauge_field(dims, C1["eps"], C1["seed"]), inputs.momentum_list(2)


def test_tsm_decomposition(orc, setup):
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    n_lp, n_hp = 5, 2
    z4 = packed_z4(dims, C1["src_seed"], n_lp)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, info = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, z4=z4, per_source=True)
        out, ps = to_np(out), to_np(ps)
        assert info["worst_resid_lp"] <= LP["rho"] and info["worst_resid_hp"] <= HP["rho"]
        assert info["iters_lp"] > 0 and info["iters_hp"] > info["iters_lp"] / n_lp and info["launches"] > 0
        # (3) oracle combiner applied to the GPU's per-source arrays
        ref = orc.tsm_combine(ps[:n_lp], ps[n_lp:])
        assert rel_l2(out, ref) <= 1e-12
        # (4) HP per-source arrays vs the oracle end to end (unique solution): error ~ cond * rho
        for r in range(n_hp):
            eta = inputs.z4_source(dims, C1["src_seed"], r)
            s_ref, _, _, st = orc.solve(eta, U, k, mu, 1e-12)
            assert st == 0
            l_ref = orc.loops_project(s_ref, eta, U, k, mu, mom, -1)
            assert rel_l2(ps[n_lp + r], l_ref) <= 100 * HP["rho"]
            # LP arrays are only O(rho_LP) close
            assert rel_l2(ps[r], l_ref) <= 20 * LP["rho"]
        # device-generated noise (counter hash) == packed noise from the host generator
        out2, _, _ = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, z4=None, seed=C1["src_seed"])
        assert np.array_equal(to_np(out2), out)
        # host-buffer entry point == device entry point
        out3, _ = ctx.tsm_estimate_host(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, z4_host=z4)
        assert np.array_equal(out3.numpy(), out)
        # gauge field uploaded from pinned host memory (stale copies repacked) + raw accumulators through the host entry
        import torch
        ctx.tm_load_gauge_host(torch.from_numpy(np.ascontiguousarray(U)).pin_memory())
        sums, _ = ctx.tsm_estimate_host(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, z4_host=z4, partial_sums=True)
        out4 = ctx.tsm_combine_sums(sums.to(ctx.tdev), n_lp, n_hp)
        assert rel_l2(to_np(out4), out) <= 1e-14


def test_tsm_identity_nlp_equals_nhp(orc, setup):
    """N_LP = N_HP with identical sources equals the plain (HP-only) estimator within 1e-10."""
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    n = 3
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, _, _ = ctx.tsm_estimate(n, n, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=C1["src_seed"])
        plain = 0
        for r in range(n):
            eta = inputs.z4_source(dims, C1["src_seed"], r)
            s, _ = ctx.tm_cg_solve(eta, k, mu, **{kk: HP[kk] for kk in ("sloppy", "outer", "recon", "rho", "max_iter", "delta")})
            plain = plain + to_np(ctx.loop_contract_project(s, eta, k, mu, mom, t.TM_F64))
        plain = plain / n
    assert rel_l2(to_np(out), plain) <= 1e-10


def test_tsm_edge_cases(setup):
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        # n_hp = 0: plain LP mean
        out, ps, _ = ctx.tsm_estimate(2, 0, k, mu, mom, LP, HP, seed=1, per_source=True)
        assert rel_l2(to_np(out), to_np(ps).mean(axis=0)) <= 1e-14
        with pytest.raises(t.TmError):
            ctx.tsm_estimate(1, 2, k, mu, mom, LP, HP, seed=1)          # n_hp > n_lp
        with pytest.raises(t.TmError):
            ctx.tsm_estimate(0, 0, k, mu, mom, LP, HP, seed=1)
        bad = dict(LP, max_iter=1)
        with pytest.raises(t.TmError) as e:
            ctx.tsm_estimate(1, 0, k, mu, mom, bad, HP, seed=1)
        assert e.value.status == t.TM_ENOCONV
        with pytest.raises(t.TmError) as e:                          # the same inside a group of sources
            ctx.tsm_estimate(3, 2, k, mu, mom, bad, HP, seed=1)
        assert e.value.status == t.TM_ENOCONV


def test_tsm_grouped_solves_equal_single_source_solves(setup):
    """Sources are solved eight (four, two, one at the ragged end) per launch by default; every per-source array must be
    bit-identical to the one-source-per-launch path (tm_set_option(TM_OPT_GROUP, 1)), for ragged N_LP / N_HP."""
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        with pytest.raises(t.TmError):
            ctx.tm_set_option(t.TM_OPT_GROUP, 3)
        with pytest.raises(t.TmError):
            ctx.tm_set_option(7, 0)
        for n_lp, n_hp, group in ((7, 3, 0), (19, 11, 0), (9, 6, 4), (5, 3, 2), (2, 1, 0)):
            ctx.tm_set_option(t.TM_OPT_GROUP, group)
            out_p, ps_p, info_p = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
            ctx.tm_set_option(t.TM_OPT_GROUP, 1)
            out_s, ps_s, info_s = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
            ctx.tm_set_option(t.TM_OPT_GROUP, 0)
            assert np.array_equal(to_np(ps_p), to_np(ps_s)), (n_lp, n_hp)
            assert info_p["iters_lp"] == info_s["iters_lp"] and info_p["iters_hp"] == info_s["iters_hp"]
            assert info_p["launches"] < info_s["launches"]
            assert rel_l2(to_np(out_p), to_np(out_s)) <= 1e-13        # lanes sum the sources in another order


def test_tsm_one_lane_equals_two_lanes(setup):
    """TM_OPT_LANES: one job in flight and two give the same per-source arrays bit for bit and the same estimate up to
    the order of the fp64 accumulation; on one lane the phase times add up to the total; automatic = one lane when the
    sources are solved 8 per launch, two for smaller groups."""
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        with pytest.raises(t.TmError):
            ctx.tm_set_option(t.TM_OPT_LANES, 3)
        ctx.tm_set_option(t.TM_OPT_LANES, 2)
        out2, ps2, info2 = ctx.tsm_estimate(19, 5, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
        ctx.tm_set_option(t.TM_OPT_LANES, 1)
        out1, ps1, info1 = ctx.tsm_estimate(19, 5, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
        ctx.tm_set_option(t.TM_OPT_LANES, 0)
        assert info2["lanes"] == 2 and info1["lanes"] == 1
        assert ctx.tsm_estimate(9, 2, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3)[2]["lanes"] == 1
        ctx.tm_set_option(t.TM_OPT_GROUP, 4)
        assert ctx.tsm_estimate(9, 2, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3)[2]["lanes"] == 2
        ctx.tm_set_option(t.TM_OPT_GROUP, 0)
        assert np.array_equal(to_np(ps1), to_np(ps2))
        assert rel_l2(to_np(out1), to_np(out2)) <= 1e-13
        assert info1["iters_lp"] == info2["iters_lp"] and info1["iters_hp"] == info2["iters_hp"]
        parts = info1["ms_lp_solve"] + info1["ms_hp_solve"] + info1["ms_contract"]
        assert abs(parts - info1["ms_total"]) <= 1e-6 * info1["ms_total"] and info1["ms_contract"] > 0


def test_tsm_merged_lp_groups(setup):
    """LP sources without an HP partner and without per-source output share one z-sum + assembly + accumulation per
    group (their x/y partial sums are added in the contraction's workspace: the later stages are linear).  The estimate
    must agree with the unmerged path (per_source=True switches merging off) within the fp32-accumulate bound of the LP
    contraction, per block, for ragged group sizes; with fp64 LP contractions nothing is merged and the two are equal
    up to the order of the fp64 accumulation."""
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        for n_lp, n_hp in ((27, 3), (16, 0), (11, 8)):
            out_m, _, info_m = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3)
            out_u, _, info_u = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
            got, ref = to_np(out_m), to_np(out_u)
            for f in (0, 1):
                for sl in (slice(0, 16), slice(16, 80)):
                    assert rel_l2(got[f, sl], ref[f, sl]) <= 1e-5, (n_lp, n_hp, f, sl)
            assert info_m["iters_lp"] == info_u["iters_lp"] and info_m["iters_hp"] == info_u["iters_hp"]
        # two jobs in flight: every lane merges in its own contraction workspace
        out_1, _, _ = ctx.tsm_estimate(43, 5, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3)
        ctx.tm_set_option(t.TM_OPT_LANES, 2)
        out_2, _, info_2 = ctx.tsm_estimate(43, 5, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3)
        ctx.tm_set_option(t.TM_OPT_LANES, 0)
        assert info_2["lanes"] == 2 and rel_l2(to_np(out_2), to_np(out_1)) <= 1e-13
        out_m, _, _ = ctx.tsm_estimate(16, 2, k, mu, mom, LP, HP, t.TM_F64, t.TM_F64, seed=3)
        out_u, _, _ = ctx.tsm_estimate(16, 2, k, mu, mom, LP, HP, t.TM_F64, t.TM_F64, seed=3, per_source=True)
        assert rel_l2(to_np(out_m), to_np(out_u)) <= 1e-13


def test_tsm_run_solutions_checked_by_oracle(orc, setup):
    """SURVEY.md sec 8 c.3 steps (1), (2) done ON the run: tsm_estimate hands back its own solutions (d_solutions) and
    the oracle evaluates, for EVERY source of a group of 8 plus a ragged tail (and both passes), the true residual
    against that source's own noise and the loops of the GPU's own s -- a mis-paired (s, eta) inside a group fails
    both.  Contractions of a given s: 1e-5 (fp32 accumulate, LP) / 1e-12 (fp64, HP) per block."""
    t = tm()
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    n_lp, n_hp = 11, 3
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, info = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=C1["src_seed"],
                                         per_source=True, solutions=True)
        ps, sol = to_np(ps), to_np(info["solutions"])
        out_plain, ps_plain, _ = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64,
                                                  seed=C1["src_seed"], per_source=True)
        assert np.array_equal(to_np(ps_plain), ps) and np.array_equal(to_np(out_plain), to_np(out))
    worst = 0.0
    for j in range(n_lp + n_hp):
        r, rho, tol = (j, LP["rho"], 1e-5) if j < n_lp else (j - n_lp, HP["rho"], 1e-12)
        eta = inputs.z4_source(dims, C1["src_seed"], r)
        true = orc.true_residual(sol[j], eta, U, k, mu, -1)
        assert true <= rho, (j, true)
        worst = max(worst, true) if j < n_lp else worst
        ref = orc.loops_project(sol[j], eta, U, k, mu, mom, -1)
        for f in (0, 1):
            for sl in (slice(0, 16), slice(16, 80)):
                assert rel_l2(ps[j][f, sl], ref[f, sl]) <= tol, (j, f, sl)
    assert abs(worst - info["worst_resid_lp"]) <= 0.05 * LP["rho"]


def test_tsm_sharded_partial_sums(orc, setup):
    """SURVEY.md sec 8e on one device: the (N_LP, N_HP) workload split round-robin over W 'ranks' (src_first = k,
    src_stride = W), each returning the raw accumulators S_LP, S_LPc, S_HP; their sum, combined by tsm_combine_sums,
    equals the single-call estimate, and every shard's per-source arrays are those of the global sources it names."""
    import torch
    t = tm()
    from paper_1401_6750_b200 import multi
    dims, U, mom = setup
    k, mu = C1["kappa"], C1["mu"]
    n_lp, n_hp = 9, 3
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, _ = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=5, per_source=True)
        ps = to_np(ps)
        for W in (2, 4):
            total = torch.zeros((3,) + tuple(out.shape), dtype=torch.complex128, device="cuda")
            for rank in range(W):
                nl, nh, first, stride = multi.shard(n_lp, n_hp, rank, W)
                sums, ps_r, _ = ctx.tsm_estimate(nl, nh, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=5, per_source=True,
                                                 src_first=first, src_stride=stride, partial_sums=True)
                ps_r, sums_h = to_np(ps_r), to_np(sums)
                glob = list(range(rank, n_lp, W))
                for j, r in enumerate(glob):
                    assert np.array_equal(ps_r[j], ps[r]), (W, rank, j)
                for j, r in enumerate(list(range(rank, n_hp, W))):
                    assert np.array_equal(ps_r[nl + j], ps[n_lp + r]), (W, rank, j)
                assert rel_l2(sums_h[0], ps_r[:nl].sum(axis=0)) <= 1e-14
                if nh:
                    assert rel_l2(sums_h[1], ps_r[:nh].sum(axis=0)) <= 1e-14
                    assert rel_l2(sums_h[2], ps_r[nl:].sum(axis=0)) <= 1e-14
                else:
                    assert not sums_h[1].any() and not sums_h[2].any()
                total += sums
            got = to_np(ctx.tsm_combine_sums(total, n_lp, n_hp))
            assert rel_l2(got, orc.tsm_combine(ps[:n_lp], ps[n_lp:])) <= 1e-12
            assert rel_l2(got, to_np(out)) <= 1e-13
