"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/pluto.h declares; without a device the compute entry points fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

from paper_2511_20337_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "pluto.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(pluto_[a-z_0-9]+)\s*\(", txt)))


def test_header_and_binding_list_the_same_symbols():
    assert _declared() == sorted(binding.SYMBOLS)


def test_library_exports_every_declared_symbol():
    L = binding.load_library()
    for name in _declared():
        assert hasattr(L, name), name


def test_argument_validation_and_no_cpu_fallback():
    import torch
    L = binding.load_library()
    assert L.pluto_workspace_bytes(1, 8, 8, 2) == 0            # nx >= 2
    assert L.pluto_workspace_bytes(8, 8, 8, 1) == 0            # ghost >= 2
    assert L.pluto_workspace_bytes(16, 16, 1, 2) > 8 * 16 * 16 * 8
    assert L.pluto_workspace_bytes(16, 16, 16, 2) > L.pluto_workspace_bytes(16, 16, 1, 2)
    if not torch.cuda.is_available():
        assert L.pluto_device_count() == 0
        assert L.pluto_init(16, 16, 1, 2, 5.0 / 3.0, 0.4, 0) == binding.ECUDA
        assert b"no CPU fallback" in L.pluto_last_error()
        assert L.pluto_step(1) == binding.ESTATE
        assert L.pluto_get_dt() != L.pluto_get_dt()            # NaN
        with pytest.raises(RuntimeError):
            binding.Pluto()


def test_oracle_and_cuda_path_share_no_code():
    """neither side includes, imports or links the other"""
    csrc = os.path.join(ROOT, "paper_2511_20337_b200")
    for root, _, files in os.walk(csrc):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h", ".py")):
                txt = open(os.path.join(root, f)).read()
                assert "oracle" not in txt.lower() or f == "workloads.py", (f, "mentions the oracle")
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".c", ".h", ".py")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "pluto.h" not in txt.replace("include/pluto.h", "") and "libpluto" not in txt and "csrc/" not in txt.replace("paper_2511_20337_b200/csrc", "")
