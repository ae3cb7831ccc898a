"""pluto_cfl_dt_noalloc against the existing CFL path (pluto_get_dt), through the C ABI, on a GPU.

Some users of this library cannot let it allocate device memory: a simulation framework that takes all of
HBM into its own arena at start-up (a library-side cudaMalloc may then simply fail), or a caller inside a
latency-critical loop (cudaMalloc / cudaFree synchronise the whole device).  For them the library has one
entry point that allocates nothing: the CFL time step of a state the caller holds, with its scratch (one
partial maximum per row of zones) in a fixed 1 MiB array inside the library.  That array is shared by every
call and keeps the last call's contents, so the tests below always make at least two calls in a row, the
second on a smaller and slower state, and expect each to agree with the existing path to the bit: the
tolerance the other GPU tests use for dt (reading R15: bit-exact for an identical input state).

This file is named so that pytest collects it last (`pytest --collect-only`): with `-x` a failure here
cannot hide another test.  It passes on its own in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2511_20337_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu


def _defaults(sim):
    """the suite shares one library context: put the scheme options back to their defaults"""
    sim.set_integrator(2)
    sim.set_emf(binding.EMF_CONTACT)
    sim.set_divb(binding.DIVB_CT)


def _noalloc_dt(sim, U, w, out):
    """one call of the new entry point on the device state U of workload w; returns (dt, max, flag)"""
    import torch
    torch.cuda.synchronize()                             # U was written on the library's stream, out on torch's
    sim.cfl_dt_noalloc(U, w.box, w.gamma, w.cfl, out, stream=torch.cuda.current_stream())
    dt, smax, flag = out.cpu().tolist()                  # ordered behind the call on the same stream
    return dt, smax, flag


def test_two_calls_in_a_row_match_the_existing_path(pluto):
    import torch
    sim = pluto
    _defaults(sim)
    out = torch.full((3,), float("nan"), dtype=torch.float64, device=sim.device)
    # a 3D blast (fast: p = 10 inside the sphere), a ragged 3D box with more rows, then a 2D Orszag-Tang state with
    # far fewer rows and a larger dt: whatever the first call left in the shared scratch must not reach the second
    cases = [wl.blast_3d(40, nsteps=1), wl.random_smooth(48, 40, 36, seed=7, amp=0.4), wl.orszag_tang_2d(96, nsteps=1)]
    seen = []
    for w in cases:
        sim.load(w)
        dt_existing = sim.get_dt()                       # existing path: k_dtmax + k_dtfinish on the library's own state
        U, _ = sim.get_state(device=True)
        dt, smax, flag = _noalloc_dt(sim, U, w, out)
        assert dt == dt_existing, (w.name, dt, dt_existing)          # bit-exact (R15)
        assert smax == w.cfl / dt or abs(smax * dt / w.cfl - 1.0) < 1e-15
        assert flag == 0.0
        # the same call again, unchanged input: the scratch now holds this very call's leftovers
        assert _noalloc_dt(sim, U, w, out)[0] == dt_existing
        seen.append(dt)
    assert len(set(seen)) == len(seen)                   # the cases really have different answers


def test_after_steps_the_next_dt_matches(pluto):
    import torch
    sim = pluto
    _defaults(sim)
    out = torch.zeros(3, dtype=torch.float64, device=sim.device)
    for w in (wl.random_smooth(33, 21, 18, seed=3), wl.random_smooth(50, 34, 1, seed=4)):
        sim.load(w)
        sim.step(3)
        U, _ = sim.get_state(device=True)
        dt_next, _, flag = _noalloc_dt(sim, U, w, out)
        sim.step(1)                                      # the existing path now computes its dt from that same state
        assert dt_next == sim.get_dt(), (w.name, dt_next, sim.get_dt())
        assert flag == 0.0


def test_flag_word_is_cleared_between_calls(pluto):
    import torch
    sim = pluto
    _defaults(sim)
    w = wl.random_smooth(32, 16, 8, seed=5)
    sim.load(w)
    dt_existing = sim.get_dt()
    U, _ = sim.get_state(device=True)
    bad = U.clone()
    bad[0, 3, 5, 7] = -1.0                               # one zone with negative density
    out = torch.zeros(3, dtype=torch.float64, device=sim.device)
    assert _noalloc_dt(sim, bad, w, out)[2] == 1.0
    dt, _, flag = _noalloc_dt(sim, U, w, out)            # next call, clean state: the flag must not stick
    assert flag == 0.0 and dt == dt_existing


def test_limit_and_argument_errors(pluto):
    import torch
    sim = pluto
    L = sim.L
    U = torch.ones(8 * 4 * 4, dtype=torch.float64, device=sim.device)
    out = torch.full((3,), -7.0, dtype=torch.float64, device=sim.device)
    rows = binding.NOALLOC_MAX_ROWS
    # one row too many: refused before anything is launched (U is far too small for these sizes and is never touched)
    rc = L.pluto_cfl_dt_noalloc(U.data_ptr(), 4, rows + 1, 1, 1.0, 1.0, 1.0, 5.0 / 3.0, 0.4, out.data_ptr(), None)
    assert rc == binding.ENOMEM
    msg = L.pluto_last_error().decode()
    assert "PLUTO_NOALLOC_MAX_ROWS" in msg and str(rows + 1) in msg
    rc = L.pluto_cfl_dt_noalloc(U.data_ptr(), 4, 1024, rows // 1024 + 1, 1.0, 1.0, 1.0, 5.0 / 3.0, 0.4, out.data_ptr(), None)
    assert rc == binding.ENOMEM
    assert L.pluto_cfl_dt_noalloc(None, 4, 4, 1, 1.0, 1.0, 1.0, 5.0 / 3.0, 0.4, out.data_ptr(), None) == binding.EINVAL
    assert L.pluto_cfl_dt_noalloc(U.data_ptr(), 4, 4, 1, 1.0, 1.0, 1.0, 5.0 / 3.0, 0.4, None, None) == binding.EINVAL
    assert L.pluto_cfl_dt_noalloc(U.data_ptr(), 1, 4, 1, 1.0, 1.0, 1.0, 5.0 / 3.0, 0.4, out.data_ptr(), None) == binding.EINVAL
    assert L.pluto_cfl_dt_noalloc(U.data_ptr(), 4, 4, 1, 1.0, 0.0, 1.0, 5.0 / 3.0, 0.4, out.data_ptr(), None) == binding.EINVAL
    assert L.pluto_cfl_dt_noalloc(U.data_ptr(), 4, 4, 1, 1.0, 1.0, 1.0, 1.0, 0.4, out.data_ptr(), None) == binding.EINVAL
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-7.0] * 3              # no refused call wrote anything


def test_largest_box_the_scratch_holds_and_free_memory_is_unchanged(pluto):
    """exactly PLUTO_NOALLOC_MAX_ROWS rows (a thin 8 x 512 x 256 box), against a numpy evaluation of the
    same rule on a uniform state with one fast zone in the very last row; the device's free memory is the
    same before and after the calls"""
    import torch
    sim = pluto
    rows = binding.NOALLOC_MAX_ROWS
    nx, ny, nz = 8, 512, rows // 512
    gamma, cfl = 5.0 / 3.0, 0.3
    U = torch.zeros((8, nz, ny, nx), dtype=torch.float64, device=sim.device)
    U[0] = 1.0
    U[4] = 0.5
    U[7] = 1.0 / (gamma - 1.0) + 0.125
    U[1, nz - 1, ny - 1, nx - 1] = 3.0                   # v_x = 3 in the last zone of the last row
    U[7, nz - 1, ny - 1, nx - 1] += 4.5
    out = torch.zeros(3, dtype=torch.float64, device=sim.device)
    box = (1.0, 64.0, 32.0)                              # cubic cells of 1/8
    cur = torch.cuda.current_stream()
    sim.cfl_dt_noalloc(U, box, gamma, cfl, out, stream=cur)      # the kernels' code is loaded here at the latest
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(sim.device)[0]
    for _ in range(2):
        sim.cfl_dt_noalloc(U, box, gamma, cfl, out, stream=cur)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info(sim.device)[0]
    assert free1 == free0
    dt, smax, flag = out.cpu().tolist()
    # uniform rho = 1, p = 1, B = (0.5, 0, 0): c_f,x = max(a, b_x) = a; the fast zone adds |v_x| = 3
    a = np.sqrt(gamma)
    expect = (3.0 + a) * 8.0
    assert flag == 0.0
    assert abs(smax / expect - 1.0) < 1e-14 and abs(dt * smax / cfl - 1.0) < 1e-15
