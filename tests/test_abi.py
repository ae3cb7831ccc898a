"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/pluto.h declares; without a device the compute entry points fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

from paper_2511_20337_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


HEADERS = ("pluto.h", "pluto_debug.h")          # the product ABI, and the test / bench entry points


def _declared(headers=HEADERS):
    names = set()
    for h in headers:
        txt = open(os.path.join(ROOT, "include", h)).read()
        txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
        names |= set(re.findall(r"\b(pluto_[a-z_0-9]+)\s*\(", txt))
    return sorted(names)


def test_product_header_holds_no_test_plumbing():
    """pluto.h is the five calls, their extensions, the slab calls and the options; counters, timers,
    the peak probe and the per-kernel debug call live in pluto_debug.h (same library)"""
    product, debug = _declared(("pluto.h",)), _declared(("pluto_debug.h",))
    assert not set(product) & set(debug)
    for name in ("pluto_init", "pluto_set_state", "pluto_step", "pluto_get_dt", "pluto_get_state", "pluto_init_slabs",
                 "pluto_set_option", "pluto_cfl_dt_noalloc"):
        assert name in product
    for name in ("pluto_debug_euler", "pluto_profile", "pluto_profile_get", "pluto_kernel_name", "pluto_launch_count",
                 "pluto_graph_captures", "pluto_probe_fp64_gflops"):
        assert name in debug and name not in product
    # both headers are plain C
    import subprocess, tempfile
    with tempfile.TemporaryDirectory() as td:
        src = os.path.join(td, "t.c")
        open(src, "w").write('#include "pluto.h"\n#include "pluto_debug.h"\nint main(void) { return PLUTO_NOALLOC_SCRATCH_BYTES > 0 ? 0 : 1; }\n')
        subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), src], check=True)


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
