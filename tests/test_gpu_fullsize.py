"""GPU parity at BASELINE.json's full size (c4: 32^3x64), in the launch configuration bench.py times.

The small-lattice tests compare every element; here the same entry points run on the paper-scale
lattice (8192 CTAs per Dslash launch, 2048 contraction CTAs, 123 momenta) and are checked
  * Dslash / full operator: every element against the oracle's fp64 apply_M (one OpenMP pass);
  * LP and HP solves with bench.py's parameters: TRUE residual by the oracle's apply_M;
  * contraction + projection: all 160 x 123 outputs of sampled timeslices against the oracle's
    direct site loop + direct DFT (the oracle computes a timeslice in a fraction of a second).
Inputs: the seeded c4 recipe, generated on the device by inputs_torch.
"""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
C4 = inputs.CONFIGS["c4"]
LP = dict(sloppy="f16", outer="f32", recon=12, rho=1e-2, max_iter=2000, delta=0.01)     # bench.py's
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=5000, delta=0.01)


@pytest.fixture(scope="module")
def c4():
    import torch
    from paper_1401_6750_b200 import inputs_torch
    t = tm()
    dev = torch.device("cuda", 0)
    dims = C4["dims"]
    U = inputs_torch.gauge_field(dims, C4["eps"], C4["seed"], dev)
    eta = inputs_torch.z4_source(dims, C4["src_seed"], 0, dev)
    ctx = t.TmContext(dims, -1, 0)
    ctx.tm_load_gauge(U)
    U_h = U.cpu().numpy()
    del U
    yield t, ctx, U_h, eta
    ctx.close()


@pytest.fixture(scope="module")
def m_ref(orc, c4):
    """Oracle M psi on a seeded Gaussian spinor (the whole 2 097 152-site lattice)."""
    import torch
    t, ctx, U_h, eta = c4
    g = torch.Generator(device="cpu")
    g.manual_seed(99)
    psi = torch.randn(tuple(eta.shape) + (2,), generator=g, dtype=torch.float64)
    psi = torch.view_as_complex(psi).numpy()
    return psi, orc.apply_M(psi, U_h, C4["kappa"], C4["mu"], -1)


@pytest.mark.parametrize("prec,recon,tol", [
    ("f64", 12, 1e-13), ("f64", 18, 1e-13), ("f32", 12, 1e-6), ("f16", 12, 5e-3), ("bf16", 12, 5e-3), ("f16", 18, 5e-3),
])
def test_operator_c4(c4, m_ref, prec, recon, tol):
    t, ctx, U_h, eta = c4
    psi, ref = m_ref
    got = to_np(ctx.apply_M(psi, C4["kappa"], C4["mu"], t.PREC[prec], recon))
    e = rel_l2(got, ref)
    assert e <= tol, (prec, recon, e)
    # the error is spread over the lattice, not concentrated on a boundary or a tile edge:
    # worst timeslice and worst z-plane stay within 2x the tolerance
    d = np.abs(got - ref) ** 2
    n = np.abs(ref) ** 2
    per_t = np.sqrt(d.sum(axis=(1, 2, 3, 4, 5)) / n.sum(axis=(1, 2, 3, 4, 5)))
    per_z = np.sqrt(d.sum(axis=(0, 2, 3, 4, 5)) / n.sum(axis=(0, 2, 3, 4, 5)))
    assert per_t.max() <= 2 * tol and per_z.max() <= 2 * tol, (per_t.max(), per_z.max())


@pytest.mark.parametrize("params", [LP, HP], ids=["lp_f16", "hp_f32_f64"])
def test_solve_c4(orc, c4, params):
    t, ctx, U_h, eta = c4
    s, info = ctx.tm_cg_solve(eta, C4["kappa"], C4["mu"], **params)
    true = orc.true_residual(to_np(s), to_np(eta), U_h, C4["kappa"], C4["mu"], -1)
    assert true <= params["rho"], (true, info)
    assert abs(info["true_resid"] - true) <= 0.05 * params["rho"]


@pytest.mark.parametrize("acc,tol", [("f32", 1e-5), ("f64", 1e-12)])
def test_contract_c4_sampled_timeslices(orc, c4, acc, tol):
    """All 160 insertions x 123 momenta on timeslices 0 (wraps to T-1), 31 and 63 (wraps to 0)."""
    t, ctx, U_h, eta = c4
    s, _ = ctx.tm_cg_solve(eta, C4["kappa"], C4["mu"], **LP)
    mom = inputs.momentum_list(9)
    got = to_np(ctx.loop_contract_project(s, eta, C4["kappa"], C4["mu"], mom, t.PREC[acc]))
    s_h, eta_h = to_np(s), to_np(eta)
    for ts in (0, 31, 63):
        ref = orc.loops_project(s_h, eta_h, U_h, C4["kappa"], C4["mu"], mom, -1, ts, ts + 1)[..., ts]
        for f in (0, 1):
            for name, sl in (("local", slice(0, 16)), ("deriv", slice(16, 80))):
                e = rel_l2(got[f, sl, :, ts], ref[f, sl])
                assert e <= tol, (acc, ts, f, name, e)


def test_tsm_c4_grouped_launches(orc, c4):
    """The launch configuration bench.py times: sources solved 8 per launch (one lane).  Per-source arrays must be
    bit-identical to the one-source-per-launch path, and a grouped solution must pass the oracle's residual check."""
    t, ctx, U_h, eta = c4
    mom = inputs.momentum_list(9)
    n_lp, n_hp = 16, 8
    ctx.tm_set_option(t.TM_OPT_GROUP, 0)
    out_g, ps_g, info_g = ctx.tsm_estimate(n_lp, n_hp, C4["kappa"], C4["mu"], mom, LP, HP, t.TM_F32, t.TM_F64,
                                           seed=C4["src_seed"], per_source=True)
    ctx.tm_set_option(t.TM_OPT_GROUP, 1)
    out_1, ps_1, info_1 = ctx.tsm_estimate(n_lp, n_hp, C4["kappa"], C4["mu"], mom, LP, HP, t.TM_F32, t.TM_F64,
                                           seed=C4["src_seed"], per_source=True)
    ctx.tm_set_option(t.TM_OPT_GROUP, 0)
    assert bool((ps_g == ps_1).all())
    assert info_g["launches"] * 4 < info_1["launches"]
    assert info_g["worst_resid_lp"] <= LP["rho"] and info_g["worst_resid_hp"] <= HP["rho"]
    assert rel_l2(to_np(out_g), to_np(out_1)) <= 1e-13
    # source 0 of the run is the fixture's eta (same seed, stream 0): its LP loops = loops of a single LP solve
    s, _ = ctx.tm_cg_solve(eta, C4["kappa"], C4["mu"], **LP)
    assert orc.true_residual(to_np(s), to_np(eta), U_h, C4["kappa"], C4["mu"], -1) <= LP["rho"]
    single = ctx.loop_contract_project(s, eta, C4["kappa"], C4["mu"], mom, t.TM_F32)
    assert rel_l2(to_np(ps_g[0]), to_np(single)) <= 1e-5


def test_tsm_c4_run_solutions_inside_a_group(orc, c4):
    """SURVEY.md sec 8 c.3 (1), (2) on the bench's launch configuration: the run's OWN solutions of sources inside a
    group of 8 (not source 0), checked by the oracle -- true residual against that source's noise, and the oracle's
    loops of the GPU's s on sampled timeslices against the run's per-source array (1e-5 fp32 / 1e-12 fp64)."""
    from paper_1401_6750_b200 import inputs_torch
    t, ctx, U_h, eta = c4
    mom = inputs.momentum_list(9)
    n_lp, n_hp = 8, 4
    _, ps, info = ctx.tsm_estimate(n_lp, n_hp, C4["kappa"], C4["mu"], mom, LP, HP, t.TM_F32, t.TM_F64,
                                   seed=C4["src_seed"], per_source=True, solutions=True)
    sol = info["solutions"]
    for j, ts in ((3, 17), (6, 63), (n_lp + 2, 0)):
        r, rho, tol = (j, LP["rho"], 1e-5) if j < n_lp else (j - n_lp, HP["rho"], 1e-12)
        eta_r = to_np(inputs_torch.z4_source(C4["dims"], C4["src_seed"], r, sol.device))
        s_h = to_np(sol[j])
        true = orc.true_residual(s_h, eta_r, U_h, C4["kappa"], C4["mu"], -1)
        assert true <= rho, (j, true)
        ref = orc.loops_project(s_h, eta_r, U_h, C4["kappa"], C4["mu"], mom, -1, ts, ts + 1)[..., ts]
        got = to_np(ps[j])
        for f in (0, 1):
            for sl in (slice(0, 16), slice(16, 80)):
                e = rel_l2(got[f, sl, :, ts], ref[f, sl])
                assert e <= tol, (j, ts, f, sl, e)
