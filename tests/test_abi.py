"""The C-ABI boundary without a GPU: libspork.so builds (nvcc cross-compiles), loads, and exports
every function include/spork.h declares; the binding declares a signature for each of them; the
struct layouts the binding mirrors have the sizes the header implies.  No compute call is made."""
import ctypes as C
import os
import re

import paper_2607_03333_b200 as sp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "spork.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # comments mention call names too
    return sorted(set(re.findall(r"\b(spork_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = sp.load()
    names = _declared()
    assert len(names) >= 30
    for n in names:
        assert hasattr(lib, n), f"libspork.so does not export {n}"
    assert sorted(sp.ABI_SYMBOLS) == names, "binding and header disagree on the ABI"
    for n in names:
        assert getattr(lib, n).argtypes is not None, f"no signature declared for {n}"


def test_struct_layouts():
    assert C.sizeof(sp.SporkConfig) == 9 * 4
    # 6 x i32, 3 x i64, 4 x i32, f32, 3 x i32
    assert C.sizeof(sp.PlanInfo) == 24 + 24 + 16 + 16
    cfg = sp.SporkConfig(sp.BF16, 32, 8, 128, 16, 64, 4, 8, 0.088)
    assert sp.load().spork_page_bytes(C.byref(cfg)) == 8 * 16 * 128 * 2
    assert sp.load().spork_strerror(sp.ERR_OOM).decode() == "out of pages"


def test_no_cpu_fallback():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        sp.Spork("bf16", 32, 8, 128, 64, 4, 8, 0.088)
