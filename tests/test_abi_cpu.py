"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/tangram.h declares, its
struct layout matches the binding, argument errors are reported before any CUDA work, and without a
device the compute calls FAIL LOUDLY (no CPU fallback).  No compute happens here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tg():
    from paper_2606_16907_b200 import build
    build.build()
    import paper_2606_16907_b200 as tg
    tg.lib()
    return tg


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tangram.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tg_[a-z_0-9]+)\s*\(", src)))


def test_exports_every_declared_symbol(tg):
    syms = declared_symbols()
    assert {"tg_instance_create", "tg_solve_batch", "tg_prune", "tg_instance_destroy"} <= set(syms)
    L = C.CDLL(tg.LIB_PATH)
    for s in syms:
        assert hasattr(L, s), f"libtangram.so does not export {s}"
    assert sorted(tg.EXPORTS) == syms, "binding and header disagree on the entry points"
    for s in syms:
        assert callable(getattr(tg, s)), f"binding lacks {s}"


def test_result_struct_layout(tg):
    assert C.sizeof(tg.TgResult) == 224 and tg.RESULT_DTYPE.itemsize == 224
    for name, _ in tg.TgResult._fields_:
        assert getattr(tg.TgResult, name).offset == tg.RESULT_DTYPE.fields[name][1]
    assert C.sizeof(tg.TgSolveStats) == 120
    assert tg.tg_version() >= 100


def test_argument_errors_need_no_device(tg):
    L = tg.lib()
    h = C.c_void_p(0)
    a = np.zeros(16, np.int32)
    p = a.ctypes.data
    assert L.tg_instance_create(2, 2, 1, 1, None, p, p, p, p, 0, C.byref(h)) == 1      # TG_ERR_NULL
    assert "NULL" in tg.tg_last_error()
    for bad in [(0, 2, 1, 1), (256, 2, 1, 1), (2, 17, 1, 1), (2, 0, 1, 1), (2, 2, 0, 1), (2, 2, 256, 1),
                (2, 2, 1, 0), (2, 2, 1, (1 << 20) + 1)]:
        assert L.tg_instance_create(*bad, p, p, p, p, p, 0, C.byref(h)) == 2           # TG_ERR_SHAPE
    assert L.tg_instance_create(2, 2, 1, 1, p, p, p, p, p, -1, C.byref(h)) == 3         # TG_ERR_RANGE
    assert h.value is None
    assert L.tg_instance_destroy(None) == 0
    assert L.tg_solve_batch(None, 0, None, None) == 0                                    # n == 0: no-op
    cnt = (C.c_int64 * 4)()
    assert L.tg_prune(None, 0, 0, cnt, None) == 1
    assert L.tg_prune_batch(None, 3, 0, 0, cnt, None) == 1
    assert L.tg_prune_batch(None, 0, 0, 0, cnt, None) == 0                               # n == 0: no-op
    assert L.tg_dp_at(None, 0, None, None) == 1
    assert L.tg_reduce(None, None, None, None, None, None, None) == 1
    assert L.tg_last_solver_kernel_ms(None) == 1
    assert L.tg_last_loader_kernel_ms(None) == 1


def test_no_cpu_fallback_without_a_device(tg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    L = tg.lib()
    h = C.c_void_p(0)
    a = np.ones(16, np.int32)
    p = a.ctypes.data
    st = L.tg_instance_create(2, 2, 1, 1, p, p, p, p, p, 0, C.byref(h))
    assert st in (4, 5) and h.value is None, "compute call must fail without CUDA"      # TG_ERR_CUDA / OOM
    with pytest.raises(tg.TangramError):
        tg.tg_instance_create(2, 2, 1, 1, a[:6], a[:6], a[:2], a[:2], a[:4], 0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_16907_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "tangram_oracle" not in txt and "oracle/" not in txt.replace("the CPU oracle", ""), f
    otxt = open(os.path.join(ROOT, "oracle", "tangram_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "#include \"../" not in otxt and "import paper_2606_16907_b200" not in otxt
