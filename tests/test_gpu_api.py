"""GPU tests of the C-ABI's call-order and life-cycle behaviour (include/pluto.h, include/pluto_debug.h): what a
rejected pluto_init leaves behind, how often a step is re-captured, what pluto_set_box does to the CFL pre-filter,
and the staged step when an option changes between its phases."""
import numpy as np
import pytest

from paper_2511_20337_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture()
def sim(pluto):
    pluto.set_integrator(2)
    pluto.set_emf(binding.EMF_CONTACT)
    pluto.set_divb(binding.DIVB_CT)
    yield pluto
    pluto.set_integrator(2)
    pluto.set_emf(binding.EMF_CONTACT)


@pytest.mark.parametrize("rk", [2, 3])
def test_one_graph_capture_for_many_single_step_calls(sim, rk):
    """a caller that steps one step per call replays the captured step; it is captured once (SSP-RK3 used to
    re-capture on every call)"""
    sim.set_integrator(rk)
    sim.load(wl.random_smooth(24, 20, 16, seed=11))
    c0 = sim.graph_captures()
    for _ in range(6):
        sim.step(1)
    sim.step_async(3)
    sim.sync()
    assert sim.graph_captures() - c0 == 1
    sim.step_fixed_dt(2, 1e-4)                           # the fixed-dt step is a second graph
    sim.step_fixed_dt(1, 1e-4)
    assert sim.graph_captures() - c0 == 2


def test_a_rejected_init_leaves_the_context_alone(sim):
    w = wl.random_smooth(20, 16, 12, seed=12)
    sim.load(w)
    sim.step(2)
    t, dt = sim.get_time(), sim.get_dt()
    U0, B0 = sim.get_state()
    L = sim.L
    assert L.pluto_init(1, 16, 12, 2, w.gamma, w.cfl, 0) == binding.EINVAL           # nx too small
    assert L.pluto_init(20, 16, 12, 2, 1.0, w.cfl, 0) == binding.EINVAL              # gamma
    assert L.pluto_init(20, 16, 12, 2, w.gamma, w.cfl, 7) == binding.EINVAL          # limiter
    assert L.pluto_init(20, 16, 12, 2, w.gamma, w.cfl, binding.WENOZ) == binding.EINVAL   # WENO-Z needs ghost >= 3
    assert L.pluto_init_slabs(5, 0, 5, 20, 16, 12, 2, w.gamma, w.cfl, 0) == binding.EINVAL    # slabs thinner than ghost + 1
    assert L.pluto_init_slabs(2, 1, 2, 20, 16, 12, 2, w.gamma, w.cfl, 0) == binding.EINVAL    # slab range
    assert L.pluto_init(256, 256, 64, 2, w.gamma, w.cfl, 0) == binding.ENOMEM        # the registered workspace is too small
    assert b"workspace" in L.pluto_last_error()
    assert sim.get_time() == t and sim.get_dt() == dt
    U1, B1 = sim.get_state()
    assert np.array_equal(U0, U1) and np.array_equal(B0, B1)
    sim.step(1)                                          # and the context still steps
    assert sim.get_time() > t


@pytest.mark.parametrize("shape", [(32, 24, 20), (48, 40, 1)])
def test_set_box_after_steps_keeps_dt_exact(sim, shape):
    """the last stage of a step leaves a grid of CFL upper bounds for the next dt reduction; they are built with
    1/dx, so pluto_set_box has to drop them (a box shrunk to a quarter: every true candidate is 4x its old bound)"""
    w = wl.blast_3d(shape[0], shape=shape, nsteps=1) if shape[2] > 1 else wl.orszag_tang_2d(shape[0], nsteps=1)
    sim.load(w)
    sim.step(3)
    U, B = sim.get_state()
    small = tuple(0.25 * l for l in w.box)
    sim.set_box(*small)
    sim.step(1)
    dt_stepped = sim.get_dt()                            # dt of the step just taken: computed after set_box
    sim.load(w)
    sim.set_box(*small)
    sim.set_state(U, B)                                  # same state, no bounds known
    assert dt_stepped == sim.get_dt()


def test_staged_step_survives_an_option_switch_between_begin_and_stage(sim):
    """pluto_step_stage makes sure of its own storage: UCT-HLLD selected after pluto_step_begin must not run the
    stage kernels on work arrays that were never allocated"""
    w = wl.random_smooth(20, 18, 16, seed=13)
    L = sim.L

    def run(switch_late):
        sim.set_emf(binding.EMF_CONTACT)
        sim.load(w, nslab=2)
        if not switch_late:
            sim.set_emf(binding.EMF_UCT_HLLD)
        assert L.pluto_step_begin(0.0) == 0
        if switch_late:
            sim.set_emf(binding.EMF_UCT_HLLD)
        for s in range(2):
            assert L.pluto_step_stage(s, 0) == 0, L.pluto_last_error()
        sim.sync()
        return sim.get_state()

    Ua, Ba = run(True)
    Ub, Bb = run(False)
    assert np.array_equal(Ua, Ub) and np.array_equal(Ba, Bb)
    assert L.pluto_step_stage(2, 0) == binding.EINVAL    # RK2 has two stages
