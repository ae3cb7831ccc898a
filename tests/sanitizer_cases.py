"""Tiny-grid driver for compute-sanitizer (SURVEY section 4(iv), section 5 "race detection").

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

Every kernel variant of the library runs at least once on a grid of a few thousand zones: the fused x+y
sweep with a whole row per block (widths 64 and 128) and in chunk mode (128- and 256-thread blocks), 2D and
3D, both limiters, the per-direction sweeps, WENO-Z, the TMA-staged and the per-thread CT kernel, RK2 and
RK3, CUDA-graph replay and plain launches, the general and the row-only ghost fill, z slabs, host and
device copies, the dt reduction with and without a bound grid, the UCT-HLLD kernels.  No oracle, no comparison: the summaries
the tool prints are kept under profiles/.
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2511_20337_b200 import workloads as wl                      # noqa: E402
from paper_2511_20337_b200.binding import OPT_CT_TMA, OPT_FUSE_XY, OPT_GRAPH, Pluto   # noqa: E402


def run(sim, w, steps=2, **kw):
    sim.load(w, **kw)
    sim.get_dt()
    sim.step(steps)
    sim.step_fixed_dt(1, 1e-4)
    sim.get_state()


def main():
    sim = Pluto(device=0)
    cases = [
        ("3D wrap 64, minmod", wl.random_smooth(64, 6, 5, seed=1, limiter=0), {}),
        ("3D wrap 128, MC", wl.random_smooth(128, 5, 4, seed=2, limiter=1), {}),
        ("3D chunk 128 (ragged)", wl.random_smooth(37, 9, 6, seed=3, limiter=0), {}),
        ("3D chunk 256 (two chunks)", wl.random_smooth(300, 5, 4, seed=4, limiter=1), {}),
        ("2D wrap 64", wl.random_smooth(64, 12, 1, seed=5, limiter=0), {}),
        ("2D chunk", wl.random_smooth(45, 17, 1, seed=6, limiter=1), {}),
        ("3D blast 16 (shock)", wl.blast_3d(16), {}),
        ("3D slabs", wl.random_smooth(40, 8, 12, seed=7, limiter=1), {"nslab": 3}),
    ]
    for name, w, kw in cases:
        for graph in (1, 0):
            sim.set_option(OPT_GRAPH, graph)
            run(sim, w, **kw)
        print("ok:", name, flush=True)
    sim.set_option(OPT_GRAPH, 1)
    # per-direction sweeps and the per-thread CT kernel
    sim.set_option(OPT_FUSE_XY, 0)
    sim.set_option(OPT_CT_TMA, 0)
    run(sim, wl.random_smooth(40, 9, 6, seed=8, limiter=1))
    run(sim, wl.random_smooth(40, 11, 1, seed=9, limiter=0))
    sim.set_option(OPT_FUSE_XY, 1)
    sim.set_option(OPT_CT_TMA, 1)
    print("ok: per-direction sweeps, per-thread CT", flush=True)
    # SSP-RK3 and WENO-Z (ghost = 3)
    sim.set_integrator(3)
    run(sim, wl.random_smooth(64, 7, 5, seed=10, limiter=1))
    for shape in ((40, 9, 7), (36, 10, 1)):
        w = wl.random_smooth(*shape, seed=11)
        w.limiter = 2
        run(sim, w)
    sim.set_integrator(2)
    print("ok: RK3, WENO-Z", flush=True)
    # UCT-HLLD EMF average (reading R19): per-direction sweeps with hlld_t<true>, k_uct_halo, k_emf_uct, k_ct_update
    sim.set_emf(1)
    run(sim, wl.random_smooth(40, 9, 6, seed=13, limiter=1))
    run(sim, wl.random_smooth(36, 11, 1, seed=14, limiter=0))
    w = wl.random_smooth(24, 9, 8, seed=15)
    w.limiter = 2
    run(sim, w)
    run(sim, wl.random_smooth(32, 8, 12, seed=16, limiter=1), nslab=2)
    sim.set_emf(0)
    print("ok: UCT-HLLD", flush=True)
    # device-pointer copies
    w = wl.random_smooth(64, 6, 5, seed=12)
    sim.load(w)
    sim.step(1)
    U, B = sim.get_state(device=True)
    sim.set_state(U, B)
    sim.step(1)
    sim.finalize()
    print("sanitizer cases done: %d launches" % sim.launch_count(), flush=True)


if __name__ == "__main__":
    main()
