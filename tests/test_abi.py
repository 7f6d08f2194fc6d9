"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/df_thermo.h declares; without a GPU the create calls fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2312_05800_b200 import build
    return build.build()


def declared_symbols():
    with open(os.path.join(ROOT, "include", "df_thermo.h")) as f:
        text = f.read()
    return sorted(set(re.findall(r"^DF_API[^;(]*?\b(df_[a-z_A-Z0-9]+)\s*\(", text, flags=re.M)))


def test_header_declares_the_hot_calls():
    syms = declared_symbols()
    for s in ("df_thermo_T_from_h", "df_thermo_properties", "df_chem_ann_source", "df_mech_create", "df_ann_create"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for s in declared_symbols():
        assert hasattr(lib, s), f"{s} declared in df_thermo.h but not exported"


def test_binding_symbol_list_matches_header(lib_path):
    from paper_2312_05800_b200 import binding
    assert sorted(binding.SYMBOLS) == declared_symbols()
    assert binding.abi_version() == 2


def test_no_cpu_fallback(lib_path):
    """On a box without a CUDA device the product path must refuse, not compute."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2312_05800_b200 import binding, synth
    with pytest.raises(binding.DfError) as e:
        binding.Mech(synth.make_mechanism(3, 1))
    assert e.value.code == binding.DF_ERR_CUDA
    with pytest.raises(binding.DfError) as e:
        binding.Ann(synth.make_ann(3, [8], 0, 1))
    assert e.value.code == binding.DF_ERR_CUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2312_05800_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, fn)) as f:
                    src = f.read()
                assert not re.search(r"^\s*(from|import)\s+oracle|#include\s+\".*oracle", src, flags=re.M), fn
