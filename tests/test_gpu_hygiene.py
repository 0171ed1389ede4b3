"""GPU memory hygiene of the CUDA path without compute-sanitizer (the tool is closed on the B200 pool this repo is
measured on, see profiles/r02_sanitizer.md): what memcheck / initcheck would flag is provoked with the library's own means.

* initcheck: TM_OPT_POISON makes every workspace the context allocates start as 0xFF bytes (NaN in fp64, fp32, fp16
  and bf16).  A kernel that reads workspace memory nothing wrote would carry NaN into the results; the runs below must
  instead be bit-identical to the same runs on zero-initialised (driver default) workspaces and finite.
* memcheck: caller-owned device buffers are carved out of a larger allocation with canaries on both sides; the canaries
  must be intact after every call that writes the buffer (operator, solver, contraction, field conversion, TSM).
* racecheck: grouped, two-lane TSM runs repeated on one context must be bit-identical run to run.
"""
import numpy as np
import pytest

from gpu_util import tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
C1 = inputs.CONFIGS["c1"]
LP = dict(sloppy="f16", outer="f32", recon=12, rho=1e-2, max_iter=500, delta=0.1)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=2000, delta=0.1)


def run_everything(t, ctx, U, dims, mom):
    """One pass over the entry points that use context workspaces; returns every result as numpy arrays."""
    k, mu = C1["kappa"], C1["mu"]
    eta = inputs.z4_source(dims, 5, 0)
    res = []
    for sloppy, outer, recon, rho in (("f64", "f64", 18, 1e-10), ("f32", "f64", 12, 1e-8), ("f16", "f32", 12, 1e-2),
                                      ("bf16", "f32", 18, 1e-2)):
        s, _ = ctx.tm_cg_solve(eta, k, mu, sloppy, outer, recon, rho)
        res.append(to_np(s))
    s = res[0]
    for acc in (t.TM_F64, t.TM_F32):
        res.append(to_np(ctx.loop_contract_project(s, eta, k, mu, mom, acc)))
        res.append(to_np(ctx.loop_contract_project_timeslice(s, eta, k, mu, mom, 3, acc)))
        res.append(to_np(ctx.loop_contract_project_explicit(s, k, mu, mom, acc)))
        res.append(to_np(ctx.loop_contract_project_sym(s, eta, k, mu, mom, acc)))
    for path in (1, 2, 3):
        ctx.tm_set_option(t.TM_OPT_CONTRACT_PATH, path)
        res.append(to_np(ctx.loop_contract_project(s, eta, k, mu, mom, t.TM_F32)))
    ctx.tm_set_option(t.TM_OPT_CONTRACT_PATH, 0)
    out, ps, _ = ctx.tsm_estimate(11, 5, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=3, per_source=True)
    res += [to_np(out), to_np(ps)]
    out, _, _ = ctx.tsm_estimate_time_diluted(2, 1, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=4)
    res.append(to_np(out))
    for prec in ("f64", "f32", "f16", "bf16"):
        res.append(to_np(ctx.apply_M(eta, k, mu, t.PREC[prec], 12)))
    return res


def test_poisoned_workspaces_change_nothing():
    t = tm()
    dims = C1["dims"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(2)
    runs = []
    for poison in (0, 1):
        with t.TmContext(dims, -1) as ctx:
            ctx.tm_set_option(t.TM_OPT_POISON, poison)
            ctx.tm_load_gauge(U)
            runs.append(run_everything(t, ctx, U, dims, mom))
    assert len(runs[0]) == len(runs[1])
    for i, (a, b) in enumerate(zip(*runs)):
        assert np.isfinite(b.view(np.float64)).all(), i
        assert np.array_equal(a, b), i
    with t.TmContext(dims, -1) as ctx:
        with pytest.raises(t.TmError):
            ctx.tm_set_option(t.TM_OPT_POISON, 2)


def guarded(torch, dev, nbytes, pad=4096):
    """A uint8 view of nbytes inside a larger allocation whose pads hold the canary value 0xA5."""
    nbytes = (nbytes + 255) // 256 * 256
    whole = torch.full((nbytes + 2 * pad,), 0xA5, dtype=torch.uint8, device=dev)
    return whole, whole[pad:pad + nbytes]


def intact(whole, pad=4096):
    return bool((whole[:pad] == 0xA5).all().item()) and bool((whole[-pad:] == 0xA5).all().item())


@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (6, 4, 6, 10), (2, 2, 2, 2)])
def test_canaries_around_caller_buffers(dims):
    """Every ABI call that writes a caller buffer, on ragged lattices (Vh not a multiple of the CTA sizes): the bytes
    right before and after the buffer must not change."""
    import torch
    t = tm()
    U = inputs.gauge_field(dims, 0.25, 13)
    mom = inputs.momentum_list(2)
    k, mu = 0.1563, 0.0055
    eta = inputs.z4_source(dims, 6, 0)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        dev = ctx.tdev
        eta_d = torch.as_tensor(eta, device=dev)
        for prec in ("f64", "f32", "f16", "bf16"):
            P = t.PREC[prec]
            fb = ctx.tm_field_bytes(P, True)
            # field import into a guarded internal field, operator into a guarded field, export into a guarded canonical
            w_in, f_in = guarded(torch, dev, fb)
            ctx._check(ctx.lib.tm_field_import(ctx.h, f_in.data_ptr(), eta_d.data_ptr(), int(P), t._stream()))
            assert intact(w_in), prec
            for recon in (12, 18):
                w_out, f_out = guarded(torch, dev, fb)
                ctx.tm_dslash(f_out, f_in, None, t.TM_OP_M_FULL, 0, False, k, mu, P, recon)
                assert intact(w_out), (prec, recon)
                pb = fb // 2
                for op in (t.TM_OP_HOP, t.TM_OP_HOP_TWINV, t.TM_OP_XPAY, t.TM_OP_MHAT):
                    w_p, f_p = guarded(torch, dev, pb)
                    ctx.tm_dslash(f_p[:pb], f_in[pb:2 * pb] if op != t.TM_OP_MHAT else f_in[:pb], f_in[:pb], op, 0, True, k, mu, P, recon)
                    assert intact(w_p), (prec, recon, op)
            w_c, c_out = guarded(torch, dev, eta_d.numel() * 16)
            ctx._check(ctx.lib.tm_field_export(ctx.h, c_out.data_ptr(), f_in.data_ptr(), int(P), t._stream()))
            assert intact(w_c), prec
        # solver output and contraction output
        nout = 160 * len(mom) * dims[3] * 16
        for acc, path in ((t.TM_F64, 0), (t.TM_F32, 1), (t.TM_F32, 2), (t.TM_F32, 3)):
            ctx.tm_set_option(t.TM_OPT_CONTRACT_PATH, path)
            s_int = ctx.tm_field_import(eta_d, acc)
            w_o, o = guarded(torch, dev, nout)
            ctx.loop_contract_project_fields(s_int, s_int, k, mu, mom, acc, out=o[:nout].view(torch.complex128))
            assert intact(w_o), (acc, path)
        ctx.tm_set_option(t.TM_OPT_CONTRACT_PATH, 0)
        torch.cuda.synchronize()


def test_grouped_two_lane_runs_repeat_bit_identically():
    """The TSM loop keeps two lanes of eight sources in flight on two streams over shared contraction tables and
    gauge copies; a data race would make repeated runs differ.  20 repetitions of a ragged run on one context."""
    t = tm()
    dims = C1["dims"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(2)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        ctx.tm_set_option(t.TM_OPT_LANES, 2)        # automatic would run groups of 8 on one lane
        first = None
        for rep in range(20):
            out, ps, _ = ctx.tsm_estimate(19, 11, C1["kappa"], C1["mu"], mom, LP, HP, t.TM_F32, t.TM_F64, seed=9, per_source=True)
            got = (to_np(out).copy(), to_np(ps).copy())
            if first is None:
                first = got
            else:
                assert np.array_equal(got[0], first[0]) and np.array_equal(got[1], first[1]), rep


def test_gauge_state_is_ordered_across_streams(orc):
    """The master gauge field is uploaded on one stream, the reduced-precision copy packed on a second and reused on a
    third, with no host synchronisation in between: the context's events must order them (include/tmloops.h,
    "Streams")."""
    import torch
    t = tm()
    c = inputs.CONFIGS["c2"]
    dims = c["dims"]
    from paper_1401_6750_b200 import inputs_torch
    dev = torch.device("cuda", 0)
    U = inputs_torch.gauge_field(dims, c["eps"], c["seed"], dev)
    U2 = inputs_torch.gauge_field(dims, c["eps"], c["seed"] + 1, dev)
    psi = inputs_torch.z4_source(dims, 3, 0, dev)
    torch.cuda.synchronize()
    s1, s2, s3 = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    with t.TmContext(dims, -1) as ctx:
        got = {}
        for name, field in (("first", U), ("second", U2)):          # the second upload overwrites a master in use
            with torch.cuda.stream(s1):
                ctx.tm_load_gauge(field)
            with torch.cuda.stream(s2):
                a = ctx.apply_M(psi, c["kappa"], c["mu"], t.TM_F32, 12)
            with torch.cuda.stream(s3):
                b = ctx.apply_M(psi, c["kappa"], c["mu"], t.TM_F32, 12)
                d = ctx.apply_M(psi, c["kappa"], c["mu"], t.TM_F64, 18)
            torch.cuda.synchronize()
            got[name] = (to_np(a), to_np(b), to_np(d))
        for name, field in (("first", U), ("second", U2)):
            ref = orc.apply_M(to_np(psi), to_np(field), c["kappa"], c["mu"], -1)
            a, b, d = got[name]
            assert np.array_equal(a, b)
            assert np.linalg.norm(a - ref) <= 1e-6 * np.linalg.norm(ref), name
            assert np.linalg.norm(d - ref) <= 1e-13 * np.linalg.norm(ref), name
