"""GPU parity: binary (power-of-two) storage of partial sums (Fig. 2)
through the C ABI vs the oracle's orc_binary_store / orc_binary_recover."""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
C1 = inputs.CONFIGS["c1"]
LP = dict(sloppy="bf16", outer="f32", recon=12, rho=1e-2, max_iter=500, delta=0.1)
HP = dict(sloppy="f32", outer="f64", recon=12, rho=1e-8, max_iter=2000, delta=0.1)


def test_accumulate_and_recover_vs_oracle(orc):
    import torch
    t = tm()
    rng = np.random.default_rng(11)
    n, shape = 15, (2, 80, 3, 8)
    ps = rng.normal(size=(n,) + shape) + 1j * rng.normal(size=(n,) + shape)
    with t.TmContext(C1["dims"], -1) as ctx:
        assert [ctx.loop_binary_nfiles(k) for k in (1, 2, 3, 4, 7, 8, 500)] == [orc.binary_nfiles(k) for k in (1, 2, 3, 4, 7, 8, 500)]
        files = torch.zeros((ctx.loop_binary_nfiles(n),) + shape, dtype=torch.complex128, device="cuda")
        d_ps = torch.from_numpy(ps).cuda()
        for stored in range(1, n + 1):
            ctx.loop_binary_accumulate(files, d_ps[stored - 1], stored - 1)
            ref_files, counts = orc.binary_store(ps[:stored])
            assert np.array_equal(to_np(files)[:len(counts)], ref_files)          # same order of additions: bit-exact
            for N in range(1, stored + 1):
                ref = orc.binary_recover(ref_files, counts, N)
                if ref is None:
                    with pytest.raises(t.TmError):
                        ctx.loop_binary_recover(files, stored, N)
                else:
                    assert rel_l2(to_np(ctx.loop_binary_recover(files, stored, N)), ref) <= 1e-15
        # Fig. 2: 13 sources = the files holding 8, 4 and 1 sources
        sel = [0] + list(range(3, 15))
        assert rel_l2(to_np(ctx.loop_binary_recover(files, n, 13)), ps[sel].mean(axis=0)) <= 1e-15
        with pytest.raises(t.TmError):
            ctx.loop_binary_recover(files, n, 16)
        # the headline run's counts: 500 sources and 20 corrections leave a partially filled last file; N = n_stored
        # recovers everything stored ("for any number of sources"), the complete prefix still works
        for n_big in (500, 20):
            big = rng.normal(size=(n_big, 2, 5)) + 1j * rng.normal(size=(n_big, 2, 5))
            d_big = torch.from_numpy(big).cuda()
            files = torch.zeros((ctx.loop_binary_nfiles(n_big), 2, 5), dtype=torch.complex128, device="cuda")
            for r in range(n_big):
                ctx.loop_binary_accumulate(files, d_big[r], r)
            ref_files, counts = orc.binary_store(big)
            assert np.array_equal(to_np(files), ref_files)
            full = 2 ** (len(counts) - 1) - 1
            for N in (n_big, full, 1):
                assert rel_l2(to_np(ctx.loop_binary_recover(files, n_big, N)), orc.binary_recover(ref_files, counts, N)) <= 1e-15
            assert rel_l2(to_np(ctx.loop_binary_recover(files, n_big, n_big)), big.mean(axis=0)) <= 1e-14
            with pytest.raises(t.TmError):
                ctx.loop_binary_recover(files, n_big, n_big - 1 if (n_big - 1) > full else full + 1)


def test_tsm_binary_partial_last_file(orc):
    """A run whose counts are not 2^K - 1 (like 500 + 20) recovers its own full estimate from the files."""
    t = tm()
    dims, k, mu = C1["dims"], C1["kappa"], C1["mu"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(1)
    n_lp, n_hp = 6, 2
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, _ = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=9, per_source=True)
        out2, f_lp, f_co, _ = ctx.tsm_estimate_binary(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=9)
        ps = to_np(ps)
        rec = to_np(ctx.loop_binary_recover(f_lp, n_lp, n_lp)) + to_np(ctx.loop_binary_recover(f_co, n_hp, n_hp))
        assert rel_l2(rec, to_np(out2)) <= 1e-13 and rel_l2(rec, to_np(out)) <= 1e-13
        assert rel_l2(rec, orc.tsm_combine(ps[:n_lp], ps[n_lp:])) <= 1e-12


def test_tsm_with_binary_files(orc):
    t = tm()
    dims, k, mu = C1["dims"], C1["kappa"], C1["mu"]
    U = inputs.gauge_field(dims, C1["eps"], C1["seed"])
    mom = inputs.momentum_list(1)
    n_lp, n_hp = 7, 3
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        out, ps, _ = ctx.tsm_estimate(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=9, per_source=True)
        out2, f_lp, f_co, _ = ctx.tsm_estimate_binary(n_lp, n_hp, k, mu, mom, LP, HP, t.TM_F32, t.TM_F64, seed=9)
        assert rel_l2(to_np(out2), to_np(out)) <= 1e-13      # one lane instead of two: another summation order
        ps = to_np(ps)
        ref_lp, c_lp = orc.binary_store(ps[:n_lp])
        ref_co, c_co = orc.binary_store(ps[n_lp:] - ps[:n_hp])
        assert list(c_lp) == [1, 2, 4] and list(c_co) == [1, 2]
        assert rel_l2(to_np(f_lp), ref_lp) <= 1e-15 and rel_l2(to_np(f_co), ref_co) <= 1e-15
        # the full TSM estimate is recoverable from the files alone ...
        rec = to_np(ctx.loop_binary_recover(f_lp, n_lp, 7)) + to_np(ctx.loop_binary_recover(f_co, n_hp, 3))
        assert rel_l2(rec, to_np(out)) <= 1e-13
        # ... and so is the estimate of a smaller run (N_LP' = 3, N_HP' = 1) = oracle combiner on those sources
        rec = to_np(ctx.loop_binary_recover(f_lp, n_lp, 3)) + to_np(ctx.loop_binary_recover(f_co, n_hp, 1))
        ref = orc.binary_recover(ref_lp, c_lp, 3) + orc.binary_recover(ref_co, c_co, 1)
        assert rel_l2(rec, ref) <= 1e-13
        direct = ps[[0, 1, 2]].mean(axis=0) + (ps[n_lp] - ps[0])
        assert rel_l2(rec, direct) <= 1e-13
