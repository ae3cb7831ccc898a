"""Build libpluto_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2511_20337_b200.build [--force]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libpluto_b200.so")
_OBJ = os.path.join(_HERE, "build")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", _INC, "-I", _CSRC]

# translation unit -> extra flags
UNITS = {
    "pluto_api.cu": [],
    "dt_kernel.cu": ["-fmad=false"],     # reading R15: the CFL expression is evaluated without contraction
}


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpluto_b200.so cannot be built (there is no CPU fallback)")


def _sources():
    out = []
    for root, _, files in os.walk(_CSRC):
        out += [os.path.join(root, f) for f in files if f.endswith((".cu", ".cuh", ".h"))]
    out += [os.path.join(_INC, "pluto.h"), os.path.join(_INC, "pluto_debug.h")]
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    """verbose: also print the ptxas resource table (-Xptxas=-v) of every kernel"""
    lib = LIB
    newest = max(os.path.getmtime(s) for s in _sources())
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
        return lib
    nvcc = _nvcc()
    objdir = _OBJ
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for unit, extra in UNITS.items():
        obj = os.path.join(objdir, unit.replace(".cu", ".o"))
        cmd = [nvcc, *ARCH, *COMMON, *extra, "-c", os.path.join(_CSRC, unit), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for cmd, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            print(out)
        if p.returncode:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    link = [nvcc, *ARCH, "-shared", "-Xcompiler", "-fPIC", "-o", lib, *objs, "-cudart", "static"]
    subprocess.run(link, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
