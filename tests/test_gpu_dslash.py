"""GPU parity: twisted-mass Dslash through the C ABI vs the CPU oracle.

Tolerances are BASELINE.json north_star's: relative L2 error of ONE application <= 1e-13 (fp64),
<= 1e-6 (fp32), <= 5e-3 (16-bit storage), measured against the fp64 oracle on UNQUANTISED inputs
(reading 12).
"""
import numpy as np
import pytest

from gpu_util import parity_mask, rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-13, "f32": 1e-6, "f16": 5e-3, "bf16": 5e-3}
C1 = inputs.CONFIGS["c1"]


@pytest.mark.parametrize("prec", ["f64", "f32", "f16", "bf16"])
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("tb", [-1, 1])
@pytest.mark.parametrize("dagger", [False, True])
def test_M_full_c1(orc, prec, recon, tb, dagger):
    t = tm()
    dims = C1["dims"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    psi = inputs.random_spinor(dims, 21)
    ref = orc.apply_M(psi, U, C1["kappa"], C1["mu"], tb, dagger)
    with t.TmContext(dims, tb) as ctx:
        ctx.tm_load_gauge(U)
        out = to_np(ctx.apply_M(psi, C1["kappa"], C1["mu"], t.PREC[prec], recon, dagger))
    assert rel_l2(out, ref) <= TOL[prec]


# several CTAs + a ragged tail (Vh = 6*4*6*10/2 = 720 = 5*128 + 80), unequal extents
@pytest.mark.parametrize("dims", [(6, 4, 6, 10), (8, 8, 8, 16), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec,recon", [("f64", 18), ("f64", 12), ("f32", 12), ("f16", 12), ("bf16", 12), ("bf16", 18)])
def test_M_full_ragged(orc, dims, prec, recon):
    t = tm()
    U = inputs.gauge_field(dims, 0.3, 31)
    psi = inputs.z4_source(dims, 32, 0) if dims[0] == 8 else inputs.random_spinor(dims, 33)
    k, mu = 0.1565, -0.02
    ref = orc.apply_M(psi, U, k, mu, -1, False)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out = to_np(ctx.apply_M(psi, k, mu, t.PREC[prec], recon, False))
    assert rel_l2(out, ref) <= TOL[prec]


def _g5(psi):
    return psi * np.array([1, 1, -1, -1]).reshape(4, 1)


def _oracle_D(orc, psi, U, tb, dagger):
    """Hopping sum from the oracle: M(mu=0) psi = psi - kappa D psi (kappa = 1)."""
    return psi - orc.apply_M(psi, U, 1.0, 0.0, tb, dagger)


@pytest.mark.parametrize("prec", ["f64", "f32", "f16", "bf16"])
@pytest.mark.parametrize("dagger", [False, True])
def test_parity_ops(orc, prec, dagger):
    """HOP, HOP_TWINV, XPAY and MHAT on one parity vs compositions of the oracle's full operator."""
    t = tm()
    dims = (4, 6, 4, 8)
    tb = -1
    k, mu = 0.156, 0.3   # large twist so a wrong twist sign is visible at 16-bit tolerance
    U = inputs.gauge_field(dims, 0.3, 41)
    psi = inputs.random_spinor(dims, 42)
    xx = inputs.random_spinor(dims, 43)
    par = parity_mask(dims)[..., None, None]
    P = t.PREC[prec]
    a = 2 * k * mu * (-1 if dagger else 1)

    def Ainv(v):
        return (v - 1j * a * _g5(v)) / (1 + a * a)

    def A(v):
        return v + 1j * a * _g5(v)

    with t.TmContext(dims, tb) as ctx:
        ctx.tm_load_gauge(U)
        fin = ctx.tm_field_import(psi, P)
        fx = ctx.tm_field_import(xx, P)
        fin_p = ctx.parity_views(fin)
        fx_p = ctx.parity_views(fx)
        for p in (0, 1):
            src = np.where(par == 1 - p, psi, 0)          # input lives on the other parity
            D = np.where(par == p, _oracle_D(orc, src, U, tb, dagger), 0)
            out = ctx.empty_field(P, True)
            out.zero_()
            op = ctx.parity_views(out)
            for name, ref in (("HOP", D), ("HOP_TWINV", Ainv(D)),
                              ("XPAY", np.where(par == p, A(xx), 0) - k * k * D)):
                ctx.tm_dslash(op[p], fin_p[1 - p], fx_p[p] if name == "XPAY" else None,
                              getattr(t, "TM_OP_" + name), p, dagger, k, mu, P, 12)
                got = to_np(ctx.tm_field_export(out, P))
                got = np.where(par == p, got, 0)
                assert rel_l2(got, ref) <= TOL[prec], (name, p)
        # Mhat x_e = A x_e - kappa^2 D_eo A^-1 D_oe x_e
        xe = np.where(par == 0, psi, 0)
        tmp = Ainv(np.where(par == 1, _oracle_D(orc, xe, U, tb, dagger), 0))
        ref = A(xe) - k * k * np.where(par == 0, _oracle_D(orc, tmp, U, tb, dagger), 0)
        out = ctx.empty_field(P, True)
        out.zero_()
        ctx.tm_dslash(ctx.parity_views(out)[0], fin_p[0], None, t.TM_OP_MHAT, 0, dagger, k, mu, P, 12)
        got = np.where(par == 0, to_np(ctx.tm_field_export(out, P)), 0)
        assert rel_l2(got, ref) <= TOL[prec]


def test_import_export_roundtrip_and_errors():
    t = tm()
    dims = (4, 4, 2, 6)
    psi = inputs.random_spinor(dims, 51)
    with t.TmContext(dims, 1) as ctx:
        f = ctx.tm_field_import(psi, t.TM_F64)
        assert np.array_equal(to_np(ctx.tm_field_export(f, t.TM_F64)), psi)
        f32 = ctx.tm_field_import(psi, t.TM_F32)
        assert rel_l2(to_np(ctx.tm_field_export(f32, t.TM_F32)), psi) < 1e-7
        # no gauge loaded -> error, not a crash
        out = ctx.empty_field(t.TM_F64, True)
        with pytest.raises(t.TmError):
            ctx.tm_dslash(out, f, None, t.TM_OP_M_FULL, 0, False, 0.1, 0.0, t.TM_F64, 18)
        with pytest.raises(t.TmError):
            ctx.tm_dslash(f, f, None, t.TM_OP_HOP, 0, False, 0.1, 0.0, t.TM_F64, 18)   # aliasing
    with pytest.raises(t.TmError):
        t.TmContext((3, 4, 4, 4))
    with pytest.raises(t.TmError):
        t.TmContext((4, 4, 4, 4), t_boundary=0)
    with pytest.raises(t.TmError) as e:                       # maximum size: rejected before anything is allocated
        t.TmContext((128, 128, 128, 256))
    assert e.value.status == t.TM_EDIM


@pytest.mark.parametrize("prec", ["f64", "f32", "f16", "bf16"])
@pytest.mark.parametrize("nb", [2, 4, 8])
def test_dslash_multi_equals_single_launches(prec, nb):
    """Row f3: nb sources per launch (links shared through L2) -- bit-identical to nb tm_dslash calls."""
    import torch
    t = tm()
    dims = (8, 8, 8, 16) if nb < 8 else (6, 4, 6, 10)
    k, mu = 0.1565, 0.004
    U = inputs.gauge_field(dims, 0.3, 3)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        P = t.PREC[prec]
        pb = ctx.tm_field_bytes(P, False)
        fields = [ctx.tm_field_import(inputs.random_spinor(dims, seed), P) for seed in range(1, nb + 1)]
        inp = torch.cat([f[:pb] for f in fields])          # even halves as inputs
        x = torch.cat([f[pb:] for f in fields])            # odd halves as the x operand
        for op in (t.TM_OP_HOP, t.TM_OP_HOP_TWINV, t.TM_OP_XPAY):
            for par in (0, 1):
                for dag in (False, True):
                    out = torch.empty_like(inp)
                    ctx.tm_dslash_multi(out, inp, x, nb, op, par, dag, k, mu, P)
                    for b in range(nb):
                        ref = torch.empty(pb, dtype=torch.uint8, device=out.device)
                        ctx.tm_dslash(ref, inp[b * pb:(b + 1) * pb], x[b * pb:(b + 1) * pb], op, par, dag, k, mu, P, 12)
                        assert bool((out[b * pb:(b + 1) * pb] == ref).all()), (prec, nb, op, par, dag, b)
        with pytest.raises(t.TmError):
            ctx.tm_dslash_multi(inp, inp, x, nb, t.TM_OP_HOP, 0, False, k, mu, P)        # out aliases in
        with pytest.raises(t.TmError):
            ctx.tm_dslash_multi(torch.empty_like(inp), inp, None, nb, t.TM_OP_XPAY, 0, False, k, mu, P)
        with pytest.raises(t.TmError):
            ctx.tm_dslash_multi(torch.empty_like(inp), inp, x, 3, t.TM_OP_HOP, 0, False, k, mu, P)
