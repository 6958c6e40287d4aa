"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/coarse_op.h declares; no compute call is made without a GPU."""
import ctypes
import os
import re

import pytest

import paper_2212_12559_b200 as cop

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "coarse_op.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(coarse_op_[a-z0-9_]+)\s*\(", src)))


def test_header_functions_match_binding_list():
    assert _declared_functions() == sorted(cop.EXPORTS)


def test_library_exports_every_declared_symbol():
    L = cop.lib()
    for name in _declared_functions():
        assert isinstance(getattr(L, name), ctypes._CFuncPtr), name


def test_null_handle_calls_are_safe_without_gpu():
    L = cop.lib()
    assert L.coarse_op_link_bytes(None) == 0
    assert L.coarse_op_scale_bytes(None) == 0
    assert L.coarse_op_vector_bytes(None, 1) == 0
    assert L.coarse_op_last_launches(None) == 0
    L.coarse_op_destroy(None)
    assert L.coarse_op_set_links(None, None, None) == cop.EINVAL
    assert "NULL" in cop.coarse_op_last_error()


def test_create_validates_before_touching_the_device():
    with pytest.raises(cop.CoarseOpError) as e:
        cop.coarse_op_create((4, 4, 4, 0), 48, cop.LINK_C64)
    assert "dims" in str(e.value)
    with pytest.raises(cop.CoarseOpError) as e:
        cop.coarse_op_create((4, 4, 4, 4), 47, cop.LINK_C64)
    assert "even" in str(e.value)


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(cop.CoarseOpError) as e:
        cop.coarse_op_create((4, 4, 4, 4), 48, cop.LINK_C64)
    assert "no CUDA device" in str(e.value)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2212_12559_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2212_12559_b200" not in text and "csrc/" not in text.replace("paper_2212_12559_b200/csrc)", "")
