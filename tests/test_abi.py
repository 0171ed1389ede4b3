"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/tmloops.h declares (no compute calls: there is no GPU here)."""
import os
import re

import paper_1401_6750_b200 as tmod
from paper_1401_6750_b200 import build as tbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "tmloops.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(?:tm_status|size_t|const char\*|long|int)\s+(\w+)\s*\(", src)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    tbuild.build()
    lib = tmod.load_library()
    decl = _declared()
    assert "tm_dslash" in decl and "tm_cg_solve" in decl and "loop_contract_project" in decl \
        and "tsm_estimate" in decl
    for name in decl:
        assert hasattr(lib, name), name
    assert sorted(tmod.EXPORTS) == decl


def test_no_cpu_fallback_without_device():
    """Without a CUDA device tm_create must fail with TM_ECUDA (never compute on the host)."""
    import torch
    if torch.cuda.is_available():
        return
    try:
        tmod.TmContext((4, 4, 4, 4))
    except tmod.TmError as e:
        assert e.status == tmod.TM_ECUDA
    else:
        raise AssertionError("tm_create succeeded without a CUDA device")


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1401_6750_b200")
    for dp, _, fns in os.walk(pkg):
        for fn in fns:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, fn
                assert "tm_oracle" not in txt and "liboracle" not in txt, fn
