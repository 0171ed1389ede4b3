"""GPU parity: eq. 2.1 solves through the C ABI vs the CPU oracle.

Bar (BASELINE.json north_star): every solve reaches a TRUE residual ||eta - M s||/||eta|| <= rho,
evaluated here by the oracle's fp64 apply_M on the exported solution (reading 8).
HP solutions are unique: they must also agree with the oracle's own 1e-12 solution to ~cond*rho.
"""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
C1 = inputs.CONFIGS["c1"]


@pytest.fixture(scope="module")
def c1(orc):
    dims = C1["dims"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    eta = inputs.z4_source(dims, C1["src_seed"], 0)
    s_ref, _, tr, st = orc.solve(eta, U, C1["kappa"], C1["mu"], 1e-12)
    assert st == 0 and tr < 2e-12
    return dims, U, eta, s_ref


@pytest.mark.parametrize("sloppy,outer,recon,rho", [
    ("f64", "f64", 18, 1e-10),      # BASELINE c1
    ("f64", "f64", 12, 1e-10),
    ("f32", "f64", 12, 1e-8),       # HP: mixed precision with reliable updates
    ("f32", "f32", 12, 1e-5),
    ("f16", "f32", 12, 1e-2),       # LP
    ("bf16", "f32", 12, 1e-2),
    ("bf16", "f32", 18, 1e-2),
    ("f16", "f64", 12, 1e-6),       # 16-bit sloppy pushed far below its own floor by reliable updates
])
def test_solve_c1(orc, c1, sloppy, outer, recon, rho):
    t = tm()
    dims, U, eta, s_ref = c1
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        s, info = ctx.tm_cg_solve(eta, C1["kappa"], C1["mu"], sloppy, outer, recon, rho, 2000)
    s = to_np(s)
    true = orc.true_residual(s, eta, U, C1["kappa"], C1["mu"], -1)
    assert true <= rho, (true, info)
    assert info["iters"] > 0
    # reported residual is honest (outer-precision evaluation of the same quantity)
    assert abs(info["true_resid"] - true) <= 0.05 * rho + 1e-6 * (outer == "f32")
    # error <= cond(M) * residual with sigma_max/sigma_min(M) ~ 20 on these fields ("<~ 20 rho";
    # measured 2.3 - 3.2 rho)
    assert rel_l2(s, s_ref) <= 20 * rho


def test_solve_medium_mixed(orc):
    """8^3x16 (several CTAs per kernel), mixed fp32/fp64 to 1e-8 and bf16 to 1e-2."""
    t = tm()
    dims = (8, 8, 8, 16)
    k, mu = 0.1565, 0.004
    U = inputs.gauge_field(dims, 0.3, 3)
    eta = inputs.z4_source(dims, 3, 1)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        for sloppy, outer, rho in (("f32", "f64", 1e-8), ("bf16", "f32", 1e-2), ("f16", "f32", 1e-2)):
            s, info = ctx.tm_cg_solve(eta, k, mu, sloppy, outer, 12, rho, 3000)
            true = orc.true_residual(to_np(s), eta, U, k, mu, -1)
            assert true <= rho, (sloppy, true, info)


def test_solve_edge_cases(orc, c1):
    t = tm()
    dims, U, eta, _ = c1
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        # zero source -> zero solution, zero iterations
        s, info = ctx.tm_cg_solve(np.zeros_like(eta), C1["kappa"], C1["mu"], "f32", "f64", 12, 1e-8, 100)
        assert np.all(to_np(s) == 0) and info["iters"] == 0
        # iteration cap -> TM_ENOCONV, solution and residual still reported
        with pytest.raises(t.TmError) as e:
            ctx.tm_cg_solve(eta, C1["kappa"], C1["mu"], "f64", "f64", 18, 1e-10, 3)
        assert e.value.status == t.TM_ENOCONV
        s, info = ctx.tm_cg_solve(eta, C1["kappa"], C1["mu"], "f64", "f64", 18, 1e-10, 3, raise_on_noconv=False)
        true = orc.true_residual(to_np(s), eta, U, C1["kappa"], C1["mu"], -1)
        assert info["status"] == t.TM_ENOCONV and info["iters"] == 3
        assert abs(info["true_resid"] - true) < 1e-10 and 1e-10 < true < 1
        # sloppy wider than outer is rejected
        with pytest.raises(t.TmError):
            ctx.tm_cg_solve(eta, C1["kappa"], C1["mu"], "f64", "f32", 18, 1e-5, 10)
        # periodic time boundary and the other flavour (mu < 0)
    with t.TmContext(dims, +1) as ctx:
        ctx.tm_load_gauge(U)
        s, info = ctx.tm_cg_solve(eta, C1["kappa"], -C1["mu"], "f32", "f64", 12, 1e-9, 2000)
        assert orc.true_residual(to_np(s), eta, U, C1["kappa"], -C1["mu"], +1) <= 1e-9


HARD = dict(dims=(16, 16, 16, 32), tb=1, eps=0.1, seed=3, kappa=0.126, mu=0.004)


def test_solve_hard_operator_16bit_reliable_updates(orc):
    """A badly conditioned operator at 16^3x32 (smooth gauge field, periodic time boundary, kappa next to the free
    critical value 1/8: the smallest singular value of M is ~ 2 kappa mu): 16-bit sloppy storage must survive several
    reliable updates -- fp16 ~100 iterations / 5 updates, bf16 ~700 iterations with the forced update every 100
    iterations -- and the mixed fp32/fp64 solve ~160 iterations.  True residuals are evaluated by the oracle."""
    import torch
    t = tm()
    from paper_1401_6750_b200 import inputs_torch
    H = HARD
    dev = torch.device("cuda", 0)
    U = inputs_torch.gauge_field(H["dims"], H["eps"], H["seed"], dev)
    eta = inputs_torch.z4_source(H["dims"], 2, 0, dev)
    U_np, eta_np = to_np(U), to_np(eta)
    with t.TmContext(H["dims"], H["tb"]) as ctx:
        ctx.tm_load_gauge(U)
        seen = {}
        for sloppy, outer, rho in (("f16", "f32", 1e-5), ("bf16", "f32", 1e-5), ("f32", "f64", 1e-8)):
            s, info = ctx.tm_cg_solve(eta, H["kappa"], H["mu"], sloppy, outer, 12, rho, 20000, 0.1)
            tr = orc.true_residual(to_np(s), eta_np, U_np, H["kappa"], H["mu"], H["tb"])
            assert tr <= rho, (sloppy, tr)
            assert abs(tr - info["true_resid"]) <= 0.05 * rho
            seen[sloppy] = info
        assert seen["f16"]["iters"] >= 60 and seen["f16"]["reliable_updates"] >= 4
        assert seen["bf16"]["iters"] >= 200 and seen["bf16"]["reliable_updates"] >= 6      # forced updates every 100
        assert seen["f32"]["iters"] >= 100 and seen["f32"]["reliable_updates"] >= 6
        # fp16 storage has no exponent range for a 1e-8 residual (unscaled vectors underflow): the solver must say so
        # (TM_ENOCONV via the stagnation rule, outputs filled) instead of iterating to max_iter or returning garbage
        s, info = ctx.tm_cg_solve(eta, H["kappa"], H["mu"], "f16", "f64", 12, 1e-8, 20000, 0.1, raise_on_noconv=False)
        assert info["status"] == t.TM_ENOCONV and info["iters"] < 2000
        tr = orc.true_residual(to_np(s), eta_np, U_np, H["kappa"], H["mu"], H["tb"])
        assert abs(tr - info["true_resid"]) <= 0.05 * max(tr, 1e-8) and tr < 1e-3


@pytest.mark.parametrize("sloppy", ["bf16", "f16"])
def test_grouped_hard_solves_pause_at_different_iterations(sloppy):
    """Eight sources of the hard operator solved in one group with 16-bit storage: they pause for reliable updates and
    finish at different iterations; every per-source array must still be bit-identical to one source per launch.
    (fp16 runs dslash16_group_kernel, where one CTA does the group's sources one after the other and the first source
    that is NOT a guarded no-op rebuilds the third link rows for the others; bf16 runs one source per CTA.)"""
    import torch
    t = tm()
    from paper_1401_6750_b200 import inputs_torch
    H = HARD
    dev = torch.device("cuda", 0)
    U = inputs_torch.gauge_field(H["dims"], H["eps"], H["seed"], dev)
    mom = inputs.momentum_list(1)
    lp = dict(sloppy=sloppy, outer="f32", recon=12, rho=1e-4, max_iter=20000, delta=0.1)
    hp = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=20000, delta=0.1)
    with t.TmContext(H["dims"], H["tb"]) as ctx:
        ctx.tm_load_gauge(U)
        out_g, ps_g, info_g = ctx.tsm_estimate(8, 2, H["kappa"], H["mu"], mom, lp, hp, t.TM_F32, t.TM_F64, seed=7, per_source=True)
        ctx.tm_set_option(t.TM_OPT_GROUP, 1)
        out_1, ps_1, info_1 = ctx.tsm_estimate(8, 2, H["kappa"], H["mu"], mom, lp, hp, t.TM_F32, t.TM_F64, seed=7, per_source=True)
        ctx.tm_set_option(t.TM_OPT_GROUP, 0)
        assert np.array_equal(to_np(ps_g), to_np(ps_1))
        assert info_g["iters_lp"] == info_1["iters_lp"] and info_g["iters_hp"] == info_1["iters_hp"]
        assert info_g["iters_lp"] >= 8 * 30 and info_g["worst_resid_lp"] <= lp["rho"] and info_g["worst_resid_hp"] <= hp["rho"]
