"""The C-ABI library loads and exports every symbol include/tno_mf.h declares; host-only entry
points behave; the product fails loudly without a GPU (no CPU fallback).  No GPU needed."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "tno_mf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tno_mf_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    import __graft_entry__
    __graft_entry__.build()
    from paper_2209_09848_b200 import binding
    lib = ctypes.CDLL(binding.LIB_PATH)
    names = _declared_functions()
    assert {"tno_mf_create", "tno_mf_search", "tno_mf_destroy", "tno_mf_inject", "tno_mf_plan",
            "tno_mf_last_error", "tno_mf_last_stats", "tno_mf_last_kernel_ms", "tno_mf_last_work",
            "tno_mf_version"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "missing export: " + n
        assert hasattr(binding, n), "binding lacks the ABI name: " + n


def test_record_sizes_match_header():
    from paper_2209_09848_b200 import binding
    assert binding.TRAJ_DTYPE.itemsize == 16          # 4 x float
    assert binding.CAND_DTYPE.itemsize == 16          # float + 3 x int32
    assert binding.SOURCE_DTYPE.itemsize == 28        # traj + 2 x int32 + float
    assert ctypes.sizeof(binding.tno_mf_config) == 48          # 9 x int32/float + one pointer, 8-byte aligned


def test_version_and_create_argument_errors():
    import paper_2209_09848_b200 as P
    assert "sm_100a" in P.tno_mf_version()
    with pytest.raises(P.TnoMfError) as e:
        P.tno_mf_create(0, None, -1, 5.0)
    assert e.value.code == -1
    with pytest.raises(P.TnoMfError) as e:
        P.tno_mf_create(0, None, 5, float("nan"))
    assert e.value.code == -1


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2209_09848_b200 as P
    with pytest.raises(P.TnoMfError) as e:
        P.tno_mf_create(0, None, 5, 5.0)
    assert e.value.code in (-3, -4)
    assert "no CPU fallback" in str(e.value) or "CUDA" in str(e.value)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2209_09848_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text and "tno_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2209_09848_b200", text, flags=re.M), f
            assert "libtno_mf" not in text and "#include \"../paper" not in text, f
