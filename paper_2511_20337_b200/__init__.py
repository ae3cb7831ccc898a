"""paper_2511_20337_b200 -- the fp64 finite-volume ideal-MHD time step of gPLUTO (arxiv 2511.20337)
as hand-written CUDA kernels for B200 (sm_100a) behind a C ABI (include/pluto.h).

    from paper_2511_20337_b200 import Pluto, workloads

`Pluto` needs the compiled library and a CUDA device; there is no CPU fallback.
"""
import importlib

from . import workloads  # noqa: F401


def __getattr__(name):
    if name in ("Pluto", "PlutoError"):
        return getattr(importlib.import_module(".binding", __name__), name)
    raise AttributeError(name)
