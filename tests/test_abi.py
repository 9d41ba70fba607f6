"""The C-ABI library loads and exports every symbol include/qdp_b200.h declares; host-side
argument validation works without a GPU.  (No compute calls here.)"""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "qdp_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qdp_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(qdp):
    names = _declared()
    assert len(names) >= 24
    lib = ctypes.CDLL(qdp.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in qdp_b200.h but not exported"
    assert sorted(qdp.DECLARED_SYMBOLS) == names, "binding and header disagree"
    for n in names:
        assert n in qdp.__all__


def test_no_device_is_an_error_not_a_fallback(qdp):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(qdp.QdpError) as e:
        qdp.qdp_lattice_create((4, 4, 4, 4))
    assert e.value.code == -8 and "no CPU fallback" in str(e.value)


def test_dims_validation_happens_before_any_device_work(qdp):
    for bad in [(3, 4, 4, 4), (4, 4, 0, 4), (4, 4, 4, 5), (1024, 1024, 64, 2)]:
        with pytest.raises(qdp.QdpError) as e:
            qdp.qdp_lattice_create(bad)
        assert e.value.code == -2
    assert qdp.qdp_kernel_launch_count() >= 0


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1111_5596_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "qdp_oracle" not in src and "orc_" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "qdp_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1111_5596_b200 import" not in osrc and "#include \"../paper" not in osrc
