"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/kratos_hydro.h declares; argument errors are reported; without a GPU the product path
fails loudly instead of falling back.  No compute calls here."""
import ctypes
import os
import re

import pytest

from paper_2501_02317_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "kratos_hydro.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kratos_hydro_[a-z0-9_]+)\s*\(", src)))


def test_header_and_binding_agree():
    assert _declared_symbols() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol():
    L = binding.load()
    for name in _declared_symbols():
        assert hasattr(L, name), name
    assert "sm_100a" in binding.version()


def test_library_is_in_tree_and_has_sm100a_code():
    path = binding.library_path()
    assert path.startswith(ROOT) and os.path.exists(path)


def _has_cuda():
    import torch
    return torch.cuda.is_available()


def test_bad_arguments_are_rejected():
    L = binding.load()
    bc = (ctypes.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert not L.kratos_hydro_create(2, 1, 1, 1.4, 0, bc)          # active axis with < 4 cells
    assert "4" in binding.last_error()
    assert not L.kratos_hydro_create(16, 1, 1, 1.0, 0, bc)         # gamma <= 1
    assert not L.kratos_hydro_create(16, 1, 1, 1.4, 3, bc)         # unknown precision
    assert not L.kratos_hydro_create(16, 1, 1, 1.4, 2 | (1 << 4), bc)   # all-fp32 state with the van Leer integrator
    bc_half = (ctypes.c_int * 6)(0, 1, 0, 0, 0, 0)
    assert not L.kratos_hydro_create(16, 1, 1, 1.4, 0, bc_half)    # periodic on one side only
    assert "periodic" in binding.last_error()
    assert L.kratos_hydro_step(None, 0.1) == binding.ERR_ARG       # NULL handle
    L.kratos_hydro_destroy(None)                                   # allowed


@pytest.mark.skipif(_has_cuda(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback_without_gpu():
    with pytest.raises(binding.KratosError) as ei:
        binding.KratosHydro(16, 16, 1, 1.4, (0,) * 6)
    assert "no CUDA device" in str(ei.value) or "CUDA" in str(ei.value)


def test_product_does_not_import_oracle():
    """The product package must never reach into oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2501_02317_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "kratos_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2501_02317_b200" not in text and "from paper_2501_02317_b200" not in text, f
            assert "kratos_hydro.h" not in text and "kh_device" not in text, f
