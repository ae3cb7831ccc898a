"""The oracle against stored values that do not come from it: SURVEY 8(c)'s independent prototype numbers,
closed forms, and its own committed regression file (tests/golden/, see the README there)."""
import math
import os

import numpy as np

from paper_2511_20337_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _read(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        if line.strip() and not line.startswith("#"):
            f = line.split()
            out[f[0]] = tuple(float(x) for x in f[1:])
    return out


def _oracle_values(oracle):
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLDEN, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return dict(mod.run())


def test_oracle_matches_the_surveys_independent_prototype(oracle):
    got = _oracle_values(oracle)
    for name, (val, rtol) in _read("survey_prototype_values.txt").items():
        assert abs(got[name] - val) <= rtol * abs(val), (name, got[name], val)


def test_oracle_regression_file_is_current(oracle):
    got = _oracle_values(oracle)
    for name, (val,) in _read("oracle_regression.txt").items():
        assert abs(got[name] - val) <= 1e-13 * abs(val), (name, got[name], val)


def test_closed_forms(oracle):
    cf = _read("closed_forms.txt")
    val, rtol = cf["blast_background_16_dt"]
    exact = 0.3 / 16.0 / math.sqrt((7.0 + math.sqrt(41.0)) / 12.0)
    assert abs(val - exact) <= 4e-16 * exact
    oracle.load(wl.blast_3d(16, noise=0.0, p_in=0.1))
    assert abs(oracle.get_dt() - exact) <= rtol * exact
    # the Alfven speed of Eq. 10's background is 1, so one wavelength is crossed in T = 1
    assert cf["cp_alfven_period"][0] == 1.0
    w = wl.cp_alfven_3d(16, noise=0.0)
    assert w.t_end == 1.0
