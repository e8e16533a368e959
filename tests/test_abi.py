"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/wslda.h
declares, sizes its workspace, and rejects bad arguments before touching a device."""
import ctypes as C
import os
import re

import paper_2602_08982_b200 as ws

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "wslda.h")).read()
    declared = sorted(set(re.findall(r"\b(wslda_[a-z_0-9]+)\s*\(", hdr)))
    assert declared, "no declarations found"
    L = ws.lib()
    for name in declared:
        assert hasattr(L, name), f"libwslda.so does not export {name}"
    assert sorted(ws.SYMBOLS) == declared


def test_workspace_bytes_is_pure_host_and_monotone():
    f = ws.make_functional(func_id=2, kin_form=1)
    a = ws.workspace_bytes((32, 32, 32), 3, 64, f)
    b = ws.workspace_bytes((32, 32, 32), 3, 4096, f)
    assert 0 < a < b                                             # grows with the per-spinor arrays
    assert ws.workspace_bytes((64, 64, 64), 3, 64, f) > ws.workspace_bytes((16, 16, 16), 3, 64, f) > 0
    assert ws.workspace_bytes((128, 32, 32), 1, 1024, f) > 0
    assert ws.workspace_bytes((64, 64, 32), 2, 128, f) > 0


def test_bad_arguments_are_rejected_on_the_host():
    f = ws.make_functional()
    assert ws.workspace_bytes((12, 8, 8), 3, 4, f) == 0          # not a power of two
    assert ws.workspace_bytes((8, 8, 8), 3, 0, f) == 0           # no spinors
    bad = ws.make_functional(ab_order=2, am_order=5)
    assert ws.workspace_bytes((8, 8, 8), 3, 4, bad) == 0
    ctx = C.c_void_p()
    d = (C.c_int * 3)(12, 8, 8)
    x = (C.c_double * 3)(1.0, 1.0, 1.0)
    rc = ws.lib().wslda_ctx_create(C.byref(ctx), d, x, 3, 4, C.byref(f), None, 0)
    assert rc == 2 and not ctx.value                             # WSLDA_EUNSUPPORTED, no launch
    d = (C.c_int * 3)(8, 8, 8)
    rc = ws.lib().wslda_ctx_create(C.byref(ctx), d, x, 3, 4, C.byref(f), None, 0)
    assert rc == 1 and b"workspace" in ws.lib().wslda_last_error(None)


def test_no_cpu_fallback():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(ws.WsldaError):
        ws.Context(3, (8, 8, 8), (1.0, 1.0, 1.0), 4)


def test_product_never_imports_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2602_08982_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "wslda_oracle" not in txt, fn


def test_bench_gpu_arm_does_not_pull_in_the_oracle_or_the_tests():
    """Importing bench.py (and building its GPU-arm helpers) must leave oracle/ and tests/ untouched: the oracle is
    imported lazily by the cpu_baseline / --impl reference legs only."""
    import subprocess
    import sys
    code = ("import sys, bench; bench.make_workload('cfg1'); "
            "bad = [m for m in sys.modules if m == 'oracle' or m.startswith('oracle.') or m == 'harness']; "
            "assert not bad, bad; assert not any(p.rstrip('/').endswith('tests') for p in sys.path), sys.path")
    subprocess.run([sys.executable, "-c", code], cwd=ROOT, check=True)
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert "import harness" not in src and "from harness" not in src and '"tests"' not in src
