"""The C-ABI library builds, loads and exports every symbol include/swept.h declares (no compute calls)."""
import ctypes
import os
import re

import pytest

import paper_1705_03162_b200 as sw

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "swept.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(swept_[a-z0-9_]+)\s*\(", text)) - {"swept_alloc_fn", "swept_free_fn"})


def test_every_declared_symbol_is_exported():
    lib = ctypes.CDLL(sw.load()._name)
    names = declared_symbols()
    assert {"swept_create", "swept_run", "swept_read", "swept_write", "swept_autotune", "swept_destroy",
            "swept_last_error", "swept_plan"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in swept.h but not exported"


def test_params_struct_matches_header():
    # 4 x 4-byte + 2 doubles + 4 pointers + 2 x 4-byte
    assert ctypes.sizeof(sw.swept_params) == 16 + 16 + 32 + 8
    assert ctypes.sizeof(sw.swept_phase) == 32  # 2 x int32, 2 x int64, 2 x int32


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(sw.SweptError):
        sw.swept_create(sw.HEAT, 2048, 1.0 / 2048, 1e-8, use_torch=False)
    with pytest.raises(sw.SweptError):
        sw.swept_create(sw.HEAT, 2048, 1.0 / 2048, 1e-8)


def test_argument_validation_without_gpu():
    with pytest.raises(sw.SweptError):
        sw.swept_create(7, 2048, 1.0, 1.0, use_torch=False)
    with pytest.raises(sw.SweptError):
        sw.swept_create(sw.HEAT, 2048, -1.0, 1.0, use_torch=False)
    assert "dx" in sw.swept_last_error()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1705_03162_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.lower() or f == "__init__.py" and "import oracle" not in txt, f
