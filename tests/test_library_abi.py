"""The C-ABI library loads on a GPU-less box and exports every symbol include/ddamg.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as entry
    entry.build()
    import paper_2407_08092_b200 as dd
    return dd.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "ddamg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ddamg_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    import paper_2407_08092_b200 as dd
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in ddamg.h but not exported"
        assert n in dd.SYMBOLS, f"{n} has no Python binding entry"
    assert sorted(dd.SYMBOLS) == names


def test_no_compute_without_gpu_and_no_cpu_fallback(lib):
    import torch
    import paper_2407_08092_b200 as dd
    assert lib.ddamg_version().startswith(b"ddamg-b200")
    h = ctypes.c_void_p()
    assert lib.ddamg_create(ctypes.byref(h), 3, 4, 1.0, 0.0, 1, 0, None) == dd.EINVAL       # odd L
    assert lib.ddamg_create(ctypes.byref(h), 4, 4, 1.0, 0.0, 7, 0, None) == dd.EINVAL       # bad bc
    assert lib.ddamg_create(None, 4, 4, 1.0, 0.0, 1, 0, None) == dd.EINVAL
    if not torch.cuda.is_available():
        assert lib.ddamg_create(ctypes.byref(h), 4, 4, 1.0, 0.0, 1, 0, None) == dd.ECUDA
        assert b"no CPU fallback" in lib.ddamg_last_error(None)
    assert lib.ddamg_destroy(None) == dd.OK
    assert lib.ddamg_apply_schur(None, None, None) == dd.EINVAL
    assert lib.ddamg_half_spinor_bytes(None) == 0


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or the other way round)."""
    pkg = os.path.join(ROOT, "paper_2407_08092_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "liboracle" not in src and "oracle/" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2407_08092_b200\b", src, flags=re.M), f
            assert "libddamg" not in src and "ddamg.h" not in src, f
