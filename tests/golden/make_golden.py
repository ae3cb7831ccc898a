#!/usr/bin/env python
"""Writes tests/golden/oracle_regression.txt.  Calls ONLY oracle/ (never the CUDA path).

    python tests/golden/make_golden.py

The values are summary statistics of oracle runs; they guard the oracle against silent drift (a change
of its arithmetic must be justified in the commit message and regenerates this file).  They are NOT the
paper's numbers: PAPER.md prints no field values ("parity unpinned").
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import Oracle                                   # noqa: E402
from paper_2511_20337_b200 import workloads as wl           # noqa: E402  (input generators only)


def run():
    o = Oracle()
    out = []
    # config 0 without noise, 100 steps
    w = wl.orszag_tang_2d(128, noise=0.0)
    o.load(w)
    out.append(("c0_nonoise_first_dt", o.get_dt()))
    assert o.step(100) == 0
    U, _ = o.get_state()
    out += [("c0_nonoise_t100", o.get_time()), ("c0_nonoise_dt100", o.get_dt()),
            ("c0_nonoise_rho_min", U[0].min()), ("c0_nonoise_rho_max", U[0].max()),
            ("c0_nonoise_mean_rho", U[0].mean()), ("c0_nonoise_mean_E", U[7].mean()),
            ("c0_nonoise_max_abs_Bx", np.abs(U[4]).max())]
    # config 1 without noise: first dt
    w = wl.cp_alfven_3d(64, noise=0.0)
    o.load(w)
    out.append(("c1_nonoise_first_dt", o.get_dt()))
    # uniform blast background 16^3, cfl 0.3: dt = cfl*dx/c_f
    w = wl.blast_3d(16, noise=0.0, p_in=0.1)
    o.load(w)
    out.append(("blast_background_16_dt", o.get_dt()))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; name value(%.17g)\n")
        for k, v in run():
            f.write(f"{k} {v:.17g}\n")
    print(open(path).read())
