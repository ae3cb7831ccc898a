"""TEST INFRASTRUCTURE ONLY -- the CPU oracle of the MHD step (see oracle/oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with paper_2511_20337_b200 (the CUDA path) and never imports it.
"""
from .binding import Oracle, build, lib_path  # noqa: F401
