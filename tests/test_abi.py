"""The C-ABI library loads without a GPU and exports every symbol include/mcrt.h declares;
without a device the entry points fail loudly (no CPU fallback).  No compute calls here."""
import ctypes
import os
import re
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1201_3588_b200 import build as B, mcrt      # noqa: E402


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "mcrt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"//[^\n]*", "", src)
    return sorted(set(re.findall(r"\b(mcrt_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def libpath():
    return B.build_library()


def test_header_symbols_all_exported(libpath):
    L = ctypes.CDLL(libpath)
    names = declared_symbols()
    assert len(names) >= 19
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/mcrt.h but not exported"
    assert sorted(mcrt.SYMBOLS) == names, "binding's symbol list and the header disagree"


def test_binding_loads_and_null_arguments_are_rejected(libpath):
    L = mcrt.lib()
    out = ctypes.c_void_p()
    assert L.mcrt_grid_create(None, ctypes.byref(out)) == -1          # MCRT_EINVAL
    assert b"NULL" in L.mcrt_last_error(None)
    assert L.mcrt_destroy(None) == -1
    assert L.mcrt_leaf_slots(None) == -1
    assert L.mcrt_run_batch(None, 1, 0, 1, None) == -1


def test_no_cpu_fallback_without_device(libpath):
    import numpy as np
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    ctx = mcrt.Context()
    with pytest.raises(mcrt.McrtError):
        ctx.grid_create(2, 0, (0, 0, 0), 1.0, None, np.ones(8, np.float32), None)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1201_3588_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "mcrt_oracle" not in txt, f
