"""GPU test of loop_contract_project_fields_static: the contraction + projection for callers that cannot allocate
(include/tmloops.h).  Its scratch lives in a file-scope device array of the library instead of context workspaces.

Checked against the existing path (loop_contract_project_fields) on the same inputs, per (f, ultra-local | derivative)
block at the tolerances of tests/test_gpu_contract.py (1e-12 fp64, 1e-5 fp32 accumulate), on two calls in a row that
use different fields AND different momentum sets (29 and 49 accumulators: another layout inside the shared array), so
that contents left by the first call cannot pass for results of the second.  Collected last on purpose (file name):
the suite runs with pytest -x.  Runs alone in a fresh process as well as after the other tests.
"""
import numpy as np
import pytest

from gpu_util import rel_l2, tm, to_np
from paper_1401_6750_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {"f64": 1e-12, "f32": 1e-5}
UNPRUNED = np.array([[3, 3, 3], [-3, 3, -2], [2, -3, 1], [0, 0, 0], [-1, -2, -3], [3, -1, 0], [1, 3, 0], [-3, -3, 0]],
                    dtype=np.int32)


def check_blocks(got, ref, tol):
    for f in (0, 1):
        for name, sl in (("local", slice(0, 16)), ("deriv", slice(16, 80))):
            e = rel_l2(got[f, sl], ref[f, sl])
            assert e <= tol, (f, name, e)


@pytest.mark.parametrize("acc", ["f64", "f32"])
@pytest.mark.parametrize("dims,tb", [((4, 4, 4, 8), -1), ((8, 6, 4, 6), 1)])
def test_static_scratch_contraction_equals_existing_path(acc, dims, tb):
    import torch
    t = tm()
    P = t.PREC[acc]
    U = inputs.gauge_field(dims, 0.3, 41)
    k, mu = 0.156, 0.01
    fields = [(inputs.random_spinor(dims, 300 + j), inputs.z4_source(dims, 400, j)) for j in range(2)]
    moms = [inputs.momentum_list(2), UNPRUNED]
    with t.TmContext(dims, tb) as ctx:
        ctx.tm_load_gauge(U)
        ints = [(ctx.tm_field_import(s, P), ctx.tm_field_import(e, P)) for s, e in fields]
        # a context that has not packed its gauge copy yet is refused (packing allocates)
        with pytest.raises(t.TmError) as ei:
            ctx.loop_contract_project_fields_static(ints[0][0], ints[0][1], k, mu, moms[0], P)
        assert ei.value.status == t.TM_EARG and "gauge" in str(ei.value)
        # existing path: reference results (this also packs the gauge copy)
        refs = [to_np(ctx.loop_contract_project_fields(si, ei_, k, mu, mom, P)) for (si, ei_), mom in zip(ints, moms)]
        outs = [torch.empty((2, 80, len(mom), dims[3]), dtype=torch.complex128, device=ctx.tdev) for mom in moms]
        # the first call on a device does the one-time set-up, and the first launch of a kernel makes the driver load
        # its code (lazy module loading): warm both kernel variants up, then the calls must not change free memory
        for j in (0, 1):
            ctx.loop_contract_project_fields_static(ints[j][0], ints[j][1], k, mu, moms[j], P, out=outs[j])
        for o in outs:
            o.fill_(float("nan"))       # (torch's own kernels load lazily too: keep them out of the measured region)
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        # two calls in a row, second one with other fields and another accumulator layout
        for j in (0, 1):
            ctx.loop_contract_project_fields_static(ints[j][0], ints[j][1], k, mu, moms[j], P, out=outs[j])
        torch.cuda.synchronize()
        # (any workspace the call allocated would take at least one 2 MiB page; 1 MiB of slack keeps unrelated driver
        # housekeeping from failing the test)
        assert torch.cuda.mem_get_info()[0] >= free0 - (1 << 20)
        for j in (0, 1):
            got = to_np(outs[j])
            assert np.isfinite(got.view(np.float64)).all()
            check_blocks(got, refs[j], TOL[acc])
        # and once more in the opposite order (the array now holds the 49-accumulator layout)
        ctx.loop_contract_project_fields_static(ints[0][0], ints[0][1], k, mu, moms[0], P, out=outs[0])
        check_blocks(to_np(outs[0]), refs[0], TOL[acc])


def test_static_scratch_limits():
    t = tm()
    assert t.load_library().loop_contract_static_scratch_bytes() == 16 << 20
    dims = (16, 16, 16, 16)         # needs 16*16*29*320*8 + 16*29*7*320*8 bytes in fp64: beyond 16 MiB
    U = inputs.gauge_field(dims, 0.3, 42)
    s = inputs.random_spinor(dims, 1)
    mom = inputs.momentum_list(1)
    with t.TmContext(dims, -1) as ctx:
        ctx.tm_load_gauge(U)
        si = ctx.tm_field_import(s, t.TM_F64)
        ctx.loop_contract_project_fields(si, si, 0.156, 0.01, mom, t.TM_F64)
        with pytest.raises(t.TmError) as ei:
            ctx.loop_contract_project_fields_static(si, si, 0.156, 0.01, mom, t.TM_F64)
        assert ei.value.status == t.TM_EDIM and "bytes" in str(ei.value)
        many = np.zeros((129, 3), dtype=np.int32)
        with pytest.raises(t.TmError) as ei:
            ctx.loop_contract_project_fields_static(si, si, 0.156, 0.01, many, t.TM_F64)
        assert ei.value.status == t.TM_EARG
