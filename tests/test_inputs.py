"""Input generators: the torch variants (used for the paper-scale configs) reproduce the numpy ones."""
import numpy as np
import torch

from paper_1401_6750_b200 import inputs, inputs_torch


def test_z4_torch_matches_numpy():
    dims = (4, 2, 6, 4)
    for r in (0, 3):
        k = inputs.z4_exponents(dims, 7, r)
        assert np.array_equal(inputs_torch.z4_packed(dims, 7, r, "cpu").numpy(), inputs.pack_z4(k))
        assert np.array_equal(inputs_torch.z4_source(dims, 7, r, "cpu").numpy(), inputs.z4_source(dims, 7, r))
    # all four values occur with about equal frequency, entries have modulus 1
    e = inputs.z4_source((8, 8, 8, 8), 1, 0)
    assert np.allclose(np.abs(e), 1)
    cnt = np.bincount(inputs.z4_exponents((8, 8, 8, 8), 1, 0), minlength=4) / e.size
    assert np.all(np.abs(cnt - 0.25) < 0.01)


def test_gauge_torch_matches_numpy_and_is_su3():
    dims = (4, 4, 2, 2)
    a = inputs.gauge_field(dims, 0.3, 5)
    b = inputs_torch.gauge_field(dims, 0.3, 5, "cpu").numpy()
    assert np.allclose(a, b, atol=1e-13)
    u = a.reshape(-1, 3, 3)
    assert np.allclose(u @ u.conj().transpose(0, 2, 1), np.eye(3), atol=1e-13)
    assert np.allclose(np.linalg.det(u), 1, atol=1e-13)


def test_momentum_list_sizes():
    assert [len(inputs.momentum_list(p)) for p in (0, 1, 4, 9)] == [1, 7, 33, 123]


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference (the CPU oracle on the host cores) on the smallest config: one JSON line with the
    keys the driver reads."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--config", "c1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "tsm_sources_per_sec" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["higher_is_better"] is True
