"""CPU-side checks of the boundary: the C-ABI library builds, loads, exports every symbol that
include/cap.h declares, and rejects bad arguments on the host before touching the GPU.
No compute calls here (there is no GPU on the CPU box)."""
import ctypes as C
import os
import re

import pytest

from paper_2607_05116_b200 import build as capbuild
from paper_2607_05116_b200 import cap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    capbuild.build()
    return cap.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "cap.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cap_[a-z_]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    syms = declared_symbols()
    assert set(cap.EXPORTS) == set(syms)
    for s in syms:
        assert hasattr(lib, s), s
    assert b"sm_100a" in lib.cap_version()


def test_workspace_query(lib):
    assert lib.cap_workspace_bytes(cap.CALL_EVAL_PLACEMENTS, 1, 65536, 128, 8, 16, 256) >= 8 * (256 * 8 + 256 * 16 + 128)
    assert lib.cap_workspace_bytes(cap.CALL_DISPATCH_LAYOUT, 1, 65536, 128, 8, 16, 0) > 0
    assert lib.cap_workspace_bytes(99, 1, 1, 1, 1, 1, 1) == 0
    assert lib.cap_workspace_bytes(cap.CALL_EVAL_PLACEMENTS, 1, 10, 0, 1, 1, 1) == 0


def test_host_side_einval_without_gpu(lib):
    bad_cfgs = [cap.gate_cfg(0, 1), cap.gate_cfg(2048, 8), cap.gate_cfg(16, 17), cap.gate_cfg(16, 0),
                cap.gate_cfg(16, 2, scoring=2), cap.gate_cfg(16, 2, n_group=3),
                cap.gate_cfg(16, 5, n_group=4, topk_group=1), cap.gate_cfg(64, 2, n_group=64, topk_group=2)]
    for cfg in bad_cfgs:
        assert lib.cap_gate_topk(None, None, 1, 4, C.byref(cfg), None, None, None, 0, None) == cap.EINVAL
    ok = cap.gate_cfg(16, 2)
    assert lib.cap_gate_topk(None, None, 1, 4, C.byref(ok), None, None, None, 0, None) == cap.EINVAL   # NULL data
    assert lib.cap_gate_topk(None, None, -1, 4, C.byref(ok), None, None, None, 0, None) == cap.EINVAL
    assert lib.cap_gate_topk(None, None, 1, 1 << 40, C.byref(ok), None, None, None, 0, None) == cap.EINVAL
    assert lib.cap_coactivation(None, None, 1, 4, 2, 16, None, None, None, 0, None) == cap.EINVAL
    topo = cap.Topology(0, 1, None, 0, 1, 1, 0)
    out = cap.EvalOut()
    assert lib.cap_eval_placements(None, None, None, 1, 4, 2, 16, None, 1, C.byref(topo), None,
                                   C.byref(out), None, 0, None) == cap.EINVAL            # D = 0
    assert lib.cap_dispatch_layout(None, None, 4, 2, 16, None, 65, None, None, None, None, 0, None) == cap.EINVAL
    assert lib.cap_validate_placements(None, 1, 1, 16, 0, None) == cap.EINVAL
    pl = lambda E, D, N, ws=None, n=0: lib.cap_coact_placement(None, None, 1, E, D, N, None, None, None, None,
                                                               None, ws, n, None)
    assert pl(6, 4, 1) == cap.EINVAL and pl(6, 3, 2) == cap.EINVAL and pl(2048, 4, 1) == cap.EINVAL
    assert pl(128, 65, 1) == cap.EINVAL and pl(16, 4, 2) == cap.EINVAL                 # NULL arrays
    assert lib.cap_coact_placement(None, None, 0, 16, 4, 2, None, None, None, None, None, None, 0,
                                   None) == cap.EWORKSPACE
    assert lib.cap_pairwise_objective(None, None, 1, 16, None, 2, None, 0.5, None, None, None, None, None) == cap.EINVAL
    assert lib.cap_pairwise_objective(None, None, 1, 16, None, 2, C.byref(topo), 0.5, None, None, None, None,
                                      None) == cap.EINVAL                                 # D = 0
    assert lib.cap_dispatch_rows(None, None, 4, 2, 16, None, 65, None, None, None, None, 0, None) == cap.EINVAL
    assert lib.cap_dispatch_rows(None, None, 4, 17, 16, None, 4, None, None, None, None, 0, None) == cap.EINVAL
    assert lib.cap_adjust_spectrum(None, None, 1, 16, 65, None, 3, None, None, None, None) == cap.EINVAL
    assert lib.cap_adjust_spectrum(None, None, 1, 16, 4, None, 3, None, None, None, None) == cap.EINVAL   # NULL arrays
    assert lib.cap_workspace_bytes(cap.CALL_DISPATCH_ROWS, 1, 65536, 128, 8, 16, 0) >= 256 * 16 * 4
    assert lib.cap_workspace_bytes(cap.CALL_COACT_PLACEMENT, 2, 0, 128, 1, 16, 0) >= 2 * 8 * (128 * 128 + 16 * 128 + 256)


def test_binding_refuses_cpu_tensors(lib):
    import torch
    with pytest.raises(cap.CapError, match="no CPU fallback"):
        cap.gate_topk(torch.zeros((1, 2, 16)), None, cap.gate_cfg(16, 2))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_05116_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "cap_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, fn
    for fn in ("cap_oracle.c", "cap_oracle.py", "build.py"):
        txt = open(os.path.join(ROOT, "oracle", fn)).read()
        assert "paper_2607_05116_b200" not in txt.replace("paper_2607_05116_b200/csrc/", ""), fn
