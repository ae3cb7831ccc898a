"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are the north_star's: fp64 max relative error <= 1e-10 after
one step, L1 relative error <= 1e-8 after 100 steps, dt bit-exact for identical input state (R15)."""
import math

import numpy as np
import pytest

from paper_2511_20337_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL_1STEP_MAXREL = 1e-10
TOL_100STEP_L1REL = 1e-8


ZERO_COMPONENT_ABS = 1e-14      # R15: a component that is identically 0 in the oracle


def _component_errors(a, b, reduce, pooled=False):
    """R15: per component  reduce|a - b| / reduce|b|  with reduce = max or sum; a component
    that is identically zero in the oracle must be <= 1e-14 absolute (returned as the second list).

    pooled=True is the explicitly named SECOND metric, used only by the 3D Orszag-Tang cases: the three
    momentum and the three field components are divided by the largest magnitude of their vector.  There
    B_z is not identically zero but ~1e-10 of |B| (it grows out of the seeded noise), so its own scale is
    far below the round-off of the vector arithmetic that produces it (|B| eps ~ 1e-16 against 1e-10)."""
    ref = [float(reduce(np.abs(b[v]))) for v in range(b.shape[0])]
    if pooled and b.shape[0] == 8:
        for grp in ((1, 2, 3), (4, 5, 6)):
            m = max(ref[v] for v in grp)
            for v in grp:
                ref[v] = m
    rel, absolute = [], []
    for v in range(a.shape[0]):
        d = float(reduce(np.abs(a[v] - b[v])))
        if ref[v] > 0:
            rel.append(d / ref[v])
        else:
            absolute.append(float(np.abs(a[v] - b[v]).max()))
    return rel, absolute


def _norm(a, b, reduce, pooled=False):
    rel, absolute = _component_errors(a, b, reduce, pooled)
    assert all(d <= ZERO_COMPONENT_ABS for d in absolute), ("component identically zero in the oracle", absolute)
    return max(rel) if rel else 0.0


def maxrel(a, b):
    """per component max|a-b| / max|b| (R15, strict: every component against its own magnitude)"""
    return _norm(a, b, np.max)


def l1rel(a, b):
    """per component sum|a-b| / sum|b| (R15, strict)"""
    return _norm(a, b, np.sum)


def maxrel_vector_scaled(a, b):
    return _norm(a, b, np.max, pooled=True)


def l1rel_vector_scaled(a, b):
    return _norm(a, b, np.sum, pooled=True)


def faces_as_components(Bf, w):
    f = wl.split_faces(Bf, w.nx, w.ny, w.nz)
    return [f[k].ravel() for k in sorted(f)]


def compare_state(pl, orc, w, tol, norm=maxrel):
    Ug, Bg = pl.get_state()
    Uo, Bo = orc.get_state()
    e_u = norm(Ug.reshape(8, -1), Uo.reshape(8, -1))
    fg, fo = faces_as_components(Bg, w), faces_as_components(Bo, w)
    e_b = max(norm(a[None], b[None]) for a, b in zip(fg, fo))
    assert e_u <= tol and e_b <= tol, (e_u, e_b)
    return e_u, e_b


SMALL = [
    ("2d_ragged_minmod", lambda: wl.random_smooth(37, 23, 1, seed=2, limiter=0, box=(1.0, 0.7, 1.0))),
    ("2d_ragged_mc", lambda: wl.random_smooth(150, 21, 1, seed=4, limiter=1)),
    ("3d_ragged_minmod", lambda: wl.random_smooth(19, 13, 11, seed=3, limiter=0, box=(1.0, 0.8, 1.1))),
    ("3d_ragged_mc", lambda: wl.random_smooth(33, 9, 14, seed=5, limiter=1)),
    ("3d_tiny", lambda: wl.random_smooth(2, 2, 2, seed=6)),
    ("2d_tiny", lambda: wl.random_smooth(2, 3, 1, seed=7)),
    ("blast_24", lambda: wl.blast_3d(24)),
    ("ot_48", lambda: wl.orszag_tang_2d(48)),
]


@pytest.mark.parametrize("name,make", SMALL, ids=[s[0] for s in SMALL])
def test_dt_is_bit_exact(pluto, oracle, name, make):
    w = make()
    pluto.load(w)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()


@pytest.mark.parametrize("name,make", SMALL, ids=[s[0] for s in SMALL])
def test_euler_stage_pieces(pluto, oracle, name, make):
    """per-kernel parity: upwind weights and induction fluxes (recon + HLLD), edge EMFs (CT average),
    then the stage output (flux-difference update, face update, cell-B mean)"""
    w = make()
    pluto.load(w)
    oracle.load(w)
    dt = oracle.get_dt()
    g = pluto.debug_euler(dt)
    o = oracle.debug_euler(dt)
    assert g["rc"] == 0 and o["rc"] == 0
    nd = 3 if w.nz > 1 else 2
    # induction fluxes kept for CT: d = x: (F_x[By], F_x[Bz]); y: (F_y[Bz], F_y[Bx]); z: (F_z[Bx], F_z[By])
    scale = np.abs(o["F"]).max()
    for d in range(nd):
        t1, t2 = (d + 1) % 3, (d + 2) % 3
        assert np.abs(g["Fem"][d, 0] - o["F"][d, 4 + t1]).max() <= 1e-12 * scale, d
        assert np.abs(g["Fem"][d, 1] - o["F"][d, 4 + t2]).max() <= 1e-12 * scale, d
        assert np.abs(g["W"][d] - o["W"][d]).max() <= 1e-9, d
    for e in range(3):
        assert np.abs(g["E"][e] - o["E"][e]).max() <= 1e-12 * max(np.abs(o["E"]).max(), 1e-300), e
    assert maxrel(g["U1"].reshape(8, -1), o["U1"].reshape(8, -1)) <= 1e-12
    assert maxrel(g["Bf1"][None], o["Bf1"][None]) <= 1e-12


@pytest.mark.parametrize("name,make", SMALL, ids=[s[0] for s in SMALL])
def test_one_step_max_rel(pluto, oracle, name, make):
    w = make()
    pluto.load(w)
    oracle.load(w)
    pluto.step(1)
    assert oracle.step(1) == 0
    assert pluto.get_dt() == oracle.get_dt()
    assert abs(pluto.get_time() - oracle.get_time()) <= 1e-15
    compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)


def test_config0_100_steps(pluto, oracle):
    """BASELINE.json configs[0]: 2D Orszag-Tang 128^2, minmod, CFL 0.4, 100 steps"""
    w = wl.config(0)
    pluto.load(w)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()
    pluto.step(1)
    oracle.step(1)
    compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
    pluto.step(99)
    assert oracle.step(99) == 0
    compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)
    assert abs(pluto.get_time() - oracle.get_time()) <= 1e-12
    # invariants on the GPU result itself
    U, Bf = pluto.get_state()
    for v in (0, 7):
        assert abs(math.fsum(U[v].ravel()) - math.fsum(w.U[v].ravel())) <= 1e-12 * abs(math.fsum(w.U[v].ravel()))
    f = wl.split_faces(Bf, w.nx, w.ny, w.nz)
    div = (f["bx"][:, :, 1:] - f["bx"][:, :, :-1]) * w.nx + (f["by"][:, 1:, :] - f["by"][:, :-1, :]) * w.ny
    assert np.abs(div).max() / w.nx <= 1e-12 * np.abs(Bf).max()
    assert np.array_equal(f["bx"][:, :, 0], f["bx"][:, :, -1]) and np.array_equal(f["by"][:, 0, :], f["by"][:, -1, :])


def _run_period(sim, w):
    t, n = 0.0, 0
    while True:
        U, Bf = sim.get_state()
        sim.set_state(U, Bf)                    # get_dt then returns the CFL dt of this state
        dt = sim.get_dt()
        if t + dt < w.t_end:
            sim.step_fixed_dt(1, dt)
            t += dt
            n += 1
        else:
            sim.step_fixed_dt(1, w.t_end - t)
            return n + 1


def test_config1_one_period(pluto, oracle):
    """configs[1]: oblique CP Alfven wave 64x32x32, MC, CFL 0.4, one period; L1 error vs exact"""
    w = wl.config(1)
    pluto.load(w)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()
    ng = _run_period(pluto, w)
    no = _run_period(oracle, w)
    assert ng == no
    compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)
    Ug, _ = pluto.get_state()
    Uo, _ = oracle.get_state()
    eg = math.sqrt(sum(np.abs(Ug[4 + s] - w.U[4 + s]).mean() ** 2 for s in range(3)))
    eo = math.sqrt(sum(np.abs(Uo[4 + s] - w.U[4 + s]).mean() ** 2 for s in range(3)))
    assert abs(eg - eo) <= 1e-9 and eg < 4e-3       # error vs the exact solution (the initial state)


def test_cfl_steps_100_3d(pluto, oracle):
    w = wl.blast_3d(32)
    pluto.load(w)
    oracle.load(w)
    pluto.step(100)
    assert oracle.step(100) == 0
    compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)


def _subbox_parity(pluto, oracle, w, centres, half=12, margin=7):
    """sampled parity at full size: the step has a finite stencil (3 cells per stage, 6 per RK2 step),
    so the oracle run on a periodic copy of a (2*half)^d sub-box with the GPU's dt reproduces the full
    run in the sub-box's core (distance > margin from its boundary)."""
    nd = w.ndim
    pluto.load(w)
    dt = pluto.get_dt()
    pluto.step(1)
    assert pluto.get_dt() == dt
    Ug, Bg = pluto.get_state()
    fg = wl.split_faces(Bg, w.nx, w.ny, w.nz)
    f0 = wl.split_faces(w.Bface, w.nx, w.ny, w.nz)
    worst = 0.0
    # momentum can be pure round-off noise in a quiet sub-box (v = 0 background of the blast): floor its
    # scale with rho * c_f of the initial data, an a-priori magnitude that does not come from either side
    rho, B2 = w.U[0], w.U[4] ** 2 + w.U[5] ** 2 + w.U[6] ** 2
    p0 = (w.gamma - 1) * (w.U[7] - 0.5 * (w.U[1] ** 2 + w.U[2] ** 2 + w.U[3] ** 2) / rho - 0.5 * B2)
    mscale = float(rho.max() * np.sqrt((w.gamma * p0.max() + B2.max()) / rho.min()))
    floor = {1: mscale, 2: mscale, 3: mscale}
    for (ci, cj, ck) in centres:
        ix = (np.arange(ci - half, ci + half)) % w.nx
        iy = (np.arange(cj - half, cj + half)) % w.ny
        iz = (np.arange(ck - half, ck + half)) % w.nz if nd == 3 else np.array([0])
        sub = lambda a: a[np.ix_(iz, iy, ix)]
        n = 2 * half
        Us = np.stack([sub(w.U[v]) for v in range(8)])
        faces = {}
        for name in ("bx", "by", "bz")[:nd]:
            a = f0[name]
            core = sub(a[:w.nz, :w.ny, :w.nx])                  # lower faces of the sub-box cells
            ax = {"bx": 2, "by": 1, "bz": 0}[name]
            faces[name] = np.concatenate([core, np.take(core, [0], axis=ax)], axis=ax)
        nzs = n if nd == 3 else 1
        assert oracle.init(n, n, nzs, 2, w.gamma, w.cfl, w.limiter) == 0
        oracle.set_box(n * w.box[0] / w.nx, n * w.box[1] / w.ny, (n * w.box[2] / w.nz) if nd == 3 else 1.0)
        oracle.set_state(Us, wl.join_faces(faces, n, n, nzs))
        assert oracle.step_fixed_dt(1, dt) == 0
        Uo, Bo = oracle.get_state()
        fo = wl.split_faces(Bo, n, n, nzs)
        c = slice(margin, n - margin)
        cz = c if nd == 3 else slice(0, 1)
        for v in range(8):
            ref = max(np.abs(Uo[v]).max(), floor.get(v, 0.0))
            d = np.abs(sub(Ug[v])[cz, c, c] - Uo[v][cz, c, c]).max()
            worst = max(worst, d / ref if ref > 0 else d)
        for name in ("bx", "by", "bz")[:nd]:
            d = np.abs(sub(fg[name][:w.nz, :w.ny, :w.nx])[cz, c, c] - fo[name][:nzs, :n, :n][cz, c, c]).max()
            worst = max(worst, d / np.abs(fo[name]).max())
    assert worst <= TOL_1STEP_MAXREL, worst
    return Ug, Bg


def test_config2_full_size_sampled(pluto, oracle):
    """configs[2]: 2D Orszag-Tang 2048^2 at full size; sub-box parity + invariants"""
    w = wl.config(2)
    rng = np.random.default_rng(0)
    centres = [(int(rng.integers(0, w.nx)), int(rng.integers(0, w.ny)), 0) for _ in range(6)] + [(0, 0, 0), (w.nx - 1, 5, 0)]
    U, Bf = _subbox_parity(pluto, oracle, w, centres)
    for v in (0, 7):
        assert abs(math.fsum(U[v].ravel()) - math.fsum(w.U[v].ravel())) <= 1e-12 * abs(math.fsum(w.U[v].ravel()))


def test_config3_full_size_sampled(pluto, oracle):
    """configs[3]: 3D blast 256^3 at full size; sub-boxes on the blast edge, at the corners, and random"""
    w = wl.config(3)
    r = int(0.1 * w.nx)
    h = w.nx // 2
    centres = [(h + r, h, h), (h, h - r, h), (h, h, h + r), (h, h, h), (0, 0, 0), (w.nx - 1, 3, w.nz - 2), (40, 200, 77)]
    U, Bf = _subbox_parity(pluto, oracle, w, centres)
    for v in (0, 7):
        assert abs(math.fsum(U[v].ravel()) - math.fsum(w.U[v].ravel())) <= 1e-12 * abs(math.fsum(w.U[v].ravel()))
    f = wl.split_faces(Bf, w.nx, w.ny, w.nz)
    div = ((f["bx"][:, :, 1:] - f["bx"][:, :, :-1]) + (f["by"][:, 1:, :] - f["by"][:, :-1, :])
           + (f["bz"][1:, :, :] - f["bz"][:-1, :, :]))
    assert np.abs(div).max() <= 1e-12 * np.abs(Bf).max()


def test_config4_full_size_sampled(pluto, oracle):
    """configs[4]: 3D blast 512^3 (134M zones, ~31 GB of library state) at full size, one step"""
    w = wl.config(4)
    r = int(0.1 * w.nx)
    h = w.nx // 2
    centres = [(h + r, h, h), (h, h, h - r), (0, 0, 0), (w.nx - 1, w.ny - 1, w.nz - 1), (100, 400, 333)]
    U, Bf = _subbox_parity(pluto, oracle, w, centres)
    for v in (0, 7):
        assert abs(math.fsum(U[v].ravel()) - math.fsum(w.U[v].ravel())) <= 1e-12 * abs(math.fsum(w.U[v].ravel()))
    pluto.finalize()


def _full_size_multi_step(pluto, oracle, w, nsteps):
    """the oracle run at FULL size next to the CUDA path, same seeded input, every element compared:
    max-rel <= 1e-10 after one step, L1-rel <= 1e-8 after `nsteps` (north_star), strict per-component R15 norm"""
    pluto.load(w)
    oracle.load(w)
    try:
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
        pluto.step(nsteps - 1)
        assert oracle.step(nsteps - 1) == 0
        e_l1 = compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)
        e_max = compare_state(pluto, oracle, w, 1e-6, norm=maxrel)      # reported; loose sanity bound only
        assert abs(pluto.get_time() - oracle.get_time()) <= 1e-10 * oracle.get_time()
        assert abs(pluto.get_dt() - oracle.get_dt()) <= 1e-10 * oracle.get_dt()
        print("\n%s: %d steps at full size: L1-rel (U, faces) = %.2e, %.2e; max-rel = %.2e, %.2e"
              % (w.name, nsteps, e_l1[0], e_l1[1], e_max[0], e_max[1]))
    finally:
        oracle.finalize()


def test_config2_full_size_100_steps(pluto, oracle):
    """configs[2] (2D Orszag-Tang 2048^2): 100 of its 200 steps, element-wise against the oracle at full size"""
    _full_size_multi_step(pluto, oracle, wl.config(2), 100)


def test_config3_full_size_50_steps(pluto, oracle):
    """configs[3] (3D blast 256^3): all 50 steps, element-wise against the oracle at full size (~10 GB host)"""
    _full_size_multi_step(pluto, oracle, wl.config(3), 50)


def test_config4_full_size_one_step_whole_domain(pluto, oracle):
    """configs[4] (3D blast 512^3): one step, every element, when the host can hold the oracle at 512^3
    (63 resident doubles per zone for RK2 = 68 GB, plus the 24 GB of input/output copies); otherwise
    test_config4_full_size_sampled (sub-boxes, one step) is the full-size evidence and DESIGN.md says so"""
    import psutil
    avail = psutil.virtual_memory().available / 2 ** 30
    if avail < 110:
        pytest.skip("host has %.0f GiB available: the 512^3 oracle needs ~95 GiB" % avail)
    w = wl.config(4)
    pluto.load(w)
    oracle.load(w)
    try:
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
    finally:
        oracle.finalize()
        pluto.finalize()


@pytest.mark.parametrize("cfg", [2, 3])
def test_dt_bit_exact_at_full_size(pluto, oracle, cfg):
    """the filtered CFL reduction returns the oracle's dt bit for bit on the full-size initial states"""
    w = wl.config(cfg)
    pluto.load(w)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()
    oracle.finalize()


def test_ct_tma_and_per_thread_paths_agree(pluto):
    """the TMA-staged CT kernel and the per-thread-load CT kernel give identical bits"""
    from paper_2511_20337_b200.binding import OPT_CT_TMA
    for shape in [(40, 24, 12), (64, 20, 1), (37, 23, 9), (31, 7, 5), (63, 15, 3)]:
        w = wl.random_smooth(*shape, seed=11, limiter=1)
        out = []
        for tma in (1, 0):
            pluto.load(w)
            pluto.set_option(OPT_CT_TMA, tma)
            pluto.step(3)
            out.append(pluto.get_state())
        pluto.set_option(OPT_CT_TMA, 1)
        assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1]), shape


def _wz(w):
    w.limiter = 2           # WENO-Z reconstruction ([51]; R18)
    return w


WENOZ_CASES = [
    ("2d_ragged", lambda: _wz(wl.random_smooth(37, 23, 1, seed=41, box=(1.0, 0.7, 1.0))), 2),
    ("2d_wide", lambda: _wz(wl.random_smooth(300, 9, 1, seed=42)), 3),
    ("3d_ragged", lambda: _wz(wl.random_smooth(19, 13, 11, seed=43, box=(1.0, 0.8, 1.1))), 3),
    ("3d_wrap_width", lambda: _wz(wl.random_smooth(64, 12, 10, seed=44)), 2),
    ("ot3d_32", lambda: _wz(wl.orszag_tang_3d(32, noise=1e-3)), 3),
]


@pytest.mark.parametrize("name,make,rk", WENOZ_CASES, ids=[s[0] for s in WENOZ_CASES])
def test_wenoz_parity(pluto, oracle, name, make, rk):
    """the paper's reconstruction (WENOZ) with RK2 and RK3: the scheme of its runs"""
    w = make()
    pluto.set_integrator(rk)
    try:
        pluto.load(w)
        oracle.load(w)
        oracle.set_integrator(rk)
        assert pluto.get_dt() == oracle.get_dt()
        # 3D Orszag-Tang: B_z is analytically zero (v_z depends on z only) and grows out of the seeded noise
        # to ~1e-10 |B|; it is compared on the scale of its vector (the named second metric of
        # _component_errors); every other case uses the strict per-component R15 norm
        n1, nl = (maxrel_vector_scaled, l1rel_vector_scaled) if name.startswith("ot3d") else (maxrel, l1rel)
        g = pluto.debug_euler(oracle.get_dt())
        o = oracle.debug_euler(oracle.get_dt())
        assert g["rc"] == 0 and o["rc"] == 0
        assert n1(g["U1"].reshape(8, -1), o["U1"].reshape(8, -1)) <= 1e-11
        assert maxrel(g["Bf1"][None], o["Bf1"][None]) <= 1e-11
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL, norm=n1)
        pluto.step(19)
        assert oracle.step(19) == 0
        compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=nl)
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


def test_wenoz_needs_three_ghost_layers(pluto):
    from paper_2511_20337_b200 import binding
    with pytest.raises(binding.PlutoError):
        pluto.init(16, 16, 16, 2, 5.0 / 3.0, 0.3, binding.WENOZ)
    pluto.init(16, 16, 16, 3, 5.0 / 3.0, 0.3, binding.WENOZ)


def test_paper_orszag_tang_3d_rk3(pluto, oracle):
    """the paper's own benchmark problem with its integrator (RK3), PLM/MC instead of WENOZ"""
    w = wl.orszag_tang_3d(32, noise=1e-3)
    pluto.set_integrator(3)
    try:
        pluto.load(w)
        oracle.load(w)
        oracle.set_integrator(3)
        assert pluto.get_dt() == oracle.get_dt()
        # B_z of this problem is noise-grown (~1e-10 |B|): vector-scaled metric, see test_wenoz_parity
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL, norm=maxrel_vector_scaled)
        pluto.step(29)
        assert oracle.step(29) == 0
        compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel_vector_scaled)
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


RK3_CASES = [
    ("2d_wrap", lambda: wl.random_smooth(64, 20, 1, seed=31, limiter=1)),
    ("2d_chunk", lambda: wl.random_smooth(150, 21, 1, seed=32, limiter=0)),
    ("3d_wrap", lambda: wl.random_smooth(64, 12, 10, seed=33, limiter=1, box=(1.0, 0.6, 0.5))),
    ("3d_ragged", lambda: wl.random_smooth(37, 23, 9, seed=34, limiter=0)),
    ("blast_24", lambda: wl.blast_3d(24)),
]


@pytest.mark.parametrize("name,make", RK3_CASES, ids=[s[0] for s in RK3_CASES])
def test_rk3_parity(pluto, oracle, name, make):
    """SSP-RK3 (Eq. 5; NEXT row 1 of SURVEY 8(f)): one step max-rel, 20 steps L1-rel"""
    w = make()
    pluto.set_integrator(3)
    try:
        pluto.load(w)
        oracle.load(w)
        assert oracle.set_integrator(3) == 0
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
        pluto.step(19)
        assert oracle.step(19) == 0
        compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)
        assert abs(pluto.get_time() - oracle.get_time()) <= 1e-12
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


@pytest.mark.parametrize("cfg", [2, 3])
def test_full_config_run_keeps_the_invariants(pluto, cfg):
    """configs[2] (200 steps) and configs[3] (50 steps) run to their full length on the GPU: mass and energy
    conserved to 1e-12, face field divergence-free to round-off, periodic duplicates equal, no unphysical zone"""
    w = wl.config(cfg)
    pluto.load(w)
    pluto.step(w.nsteps)
    U, Bf = pluto.get_state()
    assert np.isfinite(U).all() and U[0].min() > 0
    for v in (0, 7):
        tot0 = math.fsum(w.U[v].ravel())
        assert abs(math.fsum(U[v].ravel()) - tot0) <= 1e-12 * abs(tot0)
    f = wl.split_faces(Bf, w.nx, w.ny, w.nz)
    div = (f["bx"][:, :, 1:] - f["bx"][:, :, :-1]) + (f["by"][:, 1:, :] - f["by"][:, :-1, :])
    if w.nz > 1:
        div = div + (f["bz"][1:, :, :] - f["bz"][:-1, :, :])
        assert np.array_equal(f["bz"][0], f["bz"][-1])
    assert np.abs(div).max() <= 1e-12 * np.abs(Bf).max()
    assert np.array_equal(f["bx"][:, :, 0], f["bx"][:, :, -1]) and np.array_equal(f["by"][:, 0, :], f["by"][:, -1, :])


def _special_state(kind, n=(24, 16, 10), gamma=5.0 / 3.0):
    """flows that exercise the special branches of HLLD: no field at all, no normal field, a field along one
    axis only (the guarded degenerate star state), supersonic one-sided fans, exactly zero velocity"""
    nx, ny, nz = n
    base = wl.random_smooth(nx, ny, nz, seed=91, amp=0.1)
    shp = (nz, ny, nx)
    x = wl.cell_centres(nx, 1.0)[None, None, :] + np.zeros(shp)
    y = wl.cell_centres(ny, base.box[1])[None, :, None] / base.box[1] + np.zeros(shp)
    z = wl.cell_centres(nz, base.box[2])[:, None, None] / base.box[2] + np.zeros(shp)
    s2 = lambda a: np.sin(2 * np.pi * a)
    rho = 1.0 + 0.3 * s2(x) * np.cos(2 * np.pi * y)
    p = 0.6 + 0.2 * np.cos(2 * np.pi * (x + z))
    v = [0.3 * s2(y), 0.2 * s2(z), 0.1 * s2(x)]
    faces = {nm: np.zeros(sh) for nm, sh in wl.face_shapes(nx, ny, nz)}
    if kind == "hydro_supersonic":
        v = [3.0 + 0.5 * s2(y), -2.5 + 0.3 * s2(x), 2.0 * s2(x + y)]
    elif kind == "no_normal_field_x":            # B = (0, By(x), Bz(x)): B_x = 0 on every x-face, div B = 0
        faces["by"] += 0.5 + 0.2 * s2(np.broadcast_to(wl.cell_centres(nx, 1.0)[None, None, :], faces["by"].shape))
        faces["bz"] += -0.3 + 0.1 * np.cos(2 * np.pi * np.broadcast_to(wl.cell_centres(nx, 1.0)[None, None, :], faces["bz"].shape))
    elif kind == "axis_aligned_field":           # B = (1.2, 0, 0): transverse field exactly zero, c_f = c_a > a
        faces["bx"] += 1.2
        p = 0.2 + 0.05 * np.cos(2 * np.pi * x)
    elif kind == "static":
        v = [np.zeros(shp)] * 3
        faces["bx"] += 0.4; faces["by"] += -0.2; faces["bz"] += 0.7
    Bc = wl.cell_mean_of_faces(faces, nx, ny, nz, [None, None, None])
    U = wl.conserved_from_fields(rho, v, Bc, p, gamma)
    return wl.Workload(kind, nx, ny, nz, base.box, gamma, 0.3, 0, 0, U, wl.join_faces(faces, nx, ny, nz))


@pytest.mark.parametrize("kind", ["hydro_supersonic", "no_normal_field_x", "axis_aligned_field", "static"])
@pytest.mark.parametrize("lim", [0, 1])
def test_special_field_configurations(pluto, oracle, kind, lim):
    w = _special_state(kind)
    w.limiter = lim
    pluto.load(w)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()
    pluto.step(1)
    assert oracle.step(1) == 0
    compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
    pluto.step(9)
    assert oracle.step(9) == 0
    compare_state(pluto, oracle, w, TOL_100STEP_L1REL, norm=l1rel)


@pytest.mark.parametrize("lim,rk", [(0, 2), (1, 3), (2, 3)])
def test_scaled_units(pluto, oracle, lim, rk):
    """the same flow in units far from 1 (rho ~ 1e-12, p ~ 1e-8, B ~ 1e-4, v ~ 1e2, L ~ 1e10): the Newton
    reciprocals / square roots, the 1e-40 of WENO-Z and the relative guards keep the tolerances"""
    w = wl.random_smooth(40, 18, 12, seed=77, limiter=lim, amp=0.2)
    a, b, c = 1e-12, 1e-8, 1e10                      # density, pressure and length units
    vu, Bu = math.sqrt(b / a), math.sqrt(b)
    U = w.U.copy()
    U[0] *= a
    U[1:4] *= a * vu
    U[4:7] *= Bu
    U[7] *= b
    w2 = wl.Workload("scaled", w.nx, w.ny, w.nz, tuple(c * L for L in w.box), w.gamma, w.cfl, lim, 0, U, w.Bface * Bu)
    pluto.set_integrator(rk)
    try:
        pluto.load(w2)
        oracle.load(w2)
        oracle.set_integrator(rk)
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(3)
        assert oracle.step(3) == 0
        compare_state(pluto, oracle, w2, TOL_1STEP_MAXREL)
        # and it is the same flow: the unscaled run agrees to round-off after rescaling
        pluto.load(w)
        pluto.step(3)
        U1, _ = pluto.get_state()
        oracle.load(w2)
        oracle.set_integrator(rk)
        oracle.step(3)
        U2, _ = oracle.get_state()
        scale = np.array([a, a * vu, a * vu, a * vu, Bu, Bu, Bu, b]).reshape(8, 1, 1, 1)
        assert maxrel((U2 / scale).reshape(8, -1), U1.reshape(8, -1)) <= 1e-9
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


def _random_cases(count=24, seed=2024):
    rng = np.random.default_rng(seed)
    cases = []
    while len(cases) < count:
        three_d = rng.random() < 0.6
        nx = int(rng.choice([3, 5, 8, 17, 31, 32, 33, 64, 65, 100, 127, 128, 129, 200, 256, 260]))
        ny = int(rng.integers(3, 20))
        nz = int(rng.integers(3, 12)) if three_d else 1
        lim = int(rng.integers(0, 3))
        ghost = int(rng.integers(3 if lim == 2 else 2, 5))
        if min(nx, ny, nz if three_d else 99) < ghost:
            continue
        rk = int(rng.choice([2, 3]))
        box = (1.0, float(rng.uniform(0.5, 1.5)), float(rng.uniform(0.5, 1.5)))
        cases.append((nx, ny, nz, lim, ghost, rk, box, int(rng.integers(1, 10**6))))
    return cases


@pytest.mark.parametrize("case", _random_cases(), ids=lambda c: "%dx%dx%d_l%d_g%d_rk%d" % c[:6])
def test_random_shapes_two_steps(pluto, oracle, case):
    """seeded random extents (wrap widths, chunk widths, ragged tails, tiny grids), ghost counts, box shapes,
    reconstructions and integrators: two CFL steps against the oracle"""
    nx, ny, nz, lim, ghost, rk, box, seed = case
    w = wl.random_smooth(nx, ny, nz, seed=seed, limiter=lim, box=box, amp=0.15)
    pluto.set_integrator(rk)
    try:
        pluto.load(w, ghost=ghost)
        oracle.load(w)
        oracle.set_integrator(rk)
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(2)
        assert oracle.step(2) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


def test_device_pointers_and_graph_equivalence(pluto, oracle):
    """set/get with CUDA tensors; graph replay and plain launches give identical bits"""
    import torch
    from paper_2511_20337_b200 import binding
    w = wl.random_smooth(40, 24, 12, seed=9)
    pluto.load(w)
    pluto.step(3)
    U_a, B_a = pluto.get_state()
    old = pluto.set_option(binding.OPT_GRAPH, 0)
    assert old == 1
    pluto.init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter)
    pluto.set_box(*w.box)
    pluto.set_state(torch.from_numpy(w.U).cuda(), torch.from_numpy(w.Bface).cuda())
    pluto.step(3)
    U_d, B_d = pluto.get_state(device=True)
    pluto.set_option(binding.OPT_GRAPH, 1)
    assert np.array_equal(U_d.cpu().numpy(), U_a) and np.array_equal(B_d.cpu().numpy(), B_a)
    assert pluto.launch_count() > 0


@pytest.mark.parametrize("shape", [(40, 24, 12), (64, 20, 1), (37, 23, 9), (300, 9, 1), (96, 10, 6), (160, 7, 1), (192, 6, 5), (224, 5, 1)])
def test_fused_and_per_direction_sweeps_agree(pluto, shape):
    """the fused x+y sweep (wrap and chunk modes) against one kernel per direction"""
    from paper_2511_20337_b200 import binding
    w = wl.random_smooth(*shape, seed=21, limiter=1)
    pluto.load(w)
    pluto.step(2)
    Ua, Ba = pluto.get_state()
    old = pluto.set_option(binding.OPT_FUSE_XY, 0)
    try:
        pluto.load(w)
        pluto.step(2)
        Ub, Bb = pluto.get_state()
    finally:
        pluto.set_option(binding.OPT_FUSE_XY, old)
    assert maxrel(Ua.reshape(8, -1), Ub.reshape(8, -1)) <= 1e-13
    assert maxrel(Ba[None], Bb[None]) <= 1e-13


@pytest.mark.parametrize("nx,ny,nz,lim,rk", [(96, 12, 7, 0, 2), (160, 9, 1, 1, 3), (192, 8, 6, 1, 2), (224, 6, 5, 0, 3)])
def test_row_wrapping_widths_against_the_oracle(pluto, oracle, nx, ny, nz, lim, rk):
    """every multiple of 32 from 64 to 256 is an instantiated row-wide block of the fused x+y sweep (64, 128, 256
    run in the configs): the widths in between, element by element against the oracle"""
    w = wl.random_smooth(nx, ny, nz, seed=100 + nx, limiter=lim)
    pluto.set_integrator(rk)
    try:
        pluto.load(w)
        oracle.load(w)
        oracle.set_integrator(rk)
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(1)
        assert oracle.step(1) == 0
        compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)
        pluto.step(9)
        assert oracle.step(9) == 0
        compare_state(pluto, oracle, w, TOL_100STEP_L1REL)
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


def test_ghost_layers_do_not_change_the_result(pluto):
    w = wl.random_smooth(20, 18, 16, seed=12)
    pluto.load(w, ghost=2)
    pluto.step(2)
    Ua, Ba = pluto.get_state()
    pluto.load(w, ghost=4)
    pluto.step(2)
    Ub, Bb = pluto.get_state()
    assert np.array_equal(Ua, Ub) and np.array_equal(Ba, Bb)


def test_error_codes(pluto):
    from paper_2511_20337_b200 import binding
    with pytest.raises(binding.PlutoError) as e:
        pluto.init(16, 16, 1, 1)
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.PlutoError) as e:
        pluto.init(16, 16, 1, 2, gamma=1.0)
    assert e.value.code == binding.EINVAL
    w = wl.random_smooth(16, 16, 1, seed=1)
    pluto.load(w)
    with pytest.raises(binding.PlutoError) as e:
        pluto.step_fixed_dt(1, -1.0)
    assert e.value.code == binding.EINVAL
    U = w.U.copy()
    U[7, 0, 3, 3] = -5.0                           # negative pressure
    pluto.set_state(U, w.Bface)
    with pytest.raises(binding.PlutoError) as e:
        pluto.step(1)
    assert e.value.code == binding.EPHYS
    pluto.set_state(w.U, w.Bface)                   # a fresh state clears the flag
    pluto.step(1)


def test_c_abi_memory_and_call_order(pluto, oracle):
    """raw C ABI: call order errors, a too-small registered workspace, and the library's own allocation and
    stream (no torch memory, no torch stream) giving the same step as the bound path"""
    import ctypes
    import torch
    from paper_2511_20337_b200 import binding
    L = pluto.L
    w = wl.random_smooth(20, 12, 6, seed=5)
    pluto.load(w)
    pluto.step(2)
    ref = pluto.get_state()
    assert L.pluto_finalize() == 0
    assert L.pluto_step(1) == binding.ESTATE and L.pluto_get_dt() != L.pluto_get_dt()
    assert L.pluto_set_state(None, None) == binding.ESTATE
    # a registered workspace that is too small
    need = L.pluto_workspace_bytes(w.nx, w.ny, w.nz, 2)
    small = torch.empty(need // 2, dtype=torch.uint8, device="cuda")
    assert L.pluto_set_workspace(small.data_ptr(), small.numel()) == 0
    assert L.pluto_init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter) == binding.ENOMEM
    assert L.pluto_set_workspace(ctypes.c_void_p(1234567 * 256 + 8), 10) == binding.EINVAL
    # the library allocates for itself and runs on its own stream
    assert L.pluto_set_workspace(None, 0) == 0
    assert L.pluto_set_stream(None) == 0
    assert L.pluto_init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter) == 0
    assert L.pluto_set_box(*w.box) == 0
    assert L.pluto_step(1) == binding.ESTATE                      # no state yet
    U = np.ascontiguousarray(w.U)
    assert L.pluto_set_state(U.ctypes.data, w.Bface.ctypes.data) == 0
    assert L.pluto_step(2) == 0
    Uo, Bo = np.empty_like(U), np.empty_like(w.Bface)
    assert L.pluto_get_state(Uo.ctypes.data, Bo.ctypes.data) == 0
    assert np.array_equal(Uo, ref[0]) and np.array_equal(Bo, ref[1])
    assert L.pluto_get_state(None, None) == 0
    assert L.pluto_finalize() == 0
    # hand the session fixture its stream back
    assert L.pluto_set_stream(pluto.stream.cuda_stream) == 0
    pluto.workspace = None
    pluto.load(w)
    pluto.step(1)


def test_uniform_state_is_a_fixed_point(pluto):
    nx, ny, nz = 12, 10, 8
    shp = (nz, ny, nx)
    v, B = (0.4, -0.3, 0.2), (0.5, 0.8, -0.6)
    U = wl.conserved_from_fields(np.full(shp, 1.3), [np.full(shp, x) for x in v], [np.full(shp, x) for x in B],
                                 np.full(shp, 0.7), 5.0 / 3.0)
    Bf = wl.join_faces({nm: np.full(s, B["xyz".index(nm[1])]) for nm, s in wl.face_shapes(nx, ny, nz)}, nx, ny, nz)
    pluto.init(nx, ny, nz, 2, 5.0 / 3.0, 0.3, 0)
    pluto.set_state(U, Bf)
    pluto.step(3)
    U1, Bf1 = pluto.get_state()
    assert np.abs(U1 - U).max() <= 1e-15 and np.abs(Bf1 - Bf).max() <= 1e-15


# ---------------------------------------------------------------- z-slab domain decomposition

SLAB_CASES = [
    ("blast_32_chunk", lambda: wl.blast_3d(32), 2, 2),
    ("smooth_wrap64_mc", lambda: wl.random_smooth(64, 20, 26, seed=61, limiter=1, box=(1.0, 0.4, 0.5)), 2, 2),
    ("smooth_ragged_rk3", lambda: wl.random_smooth(37, 23, 19, seed=62, limiter=0), 3, 2),
    ("ot3d_wenoz_rk3", lambda: _wz(wl.orszag_tang_3d(32, noise=1e-3)), 3, 3),
]


@pytest.mark.parametrize("nslab", [2, 4])
@pytest.mark.parametrize("name,make,rk,ghost", SLAB_CASES, ids=[s[0] for s in SLAB_CASES])
def test_slabs_match_the_single_domain_bit_for_bit(pluto, name, make, rk, ghost, nslab):
    """the box cut into z slabs (ghost planes pulled from the neighbour slab, one max for dt: section 3.4,
    PAPER.md:208-244) advances exactly like the periodic single domain: same bits after 4 steps, same dt"""
    w = make()
    if w.nz // nslab < ghost + 1:
        pytest.skip("slab thinner than ghost + 1 planes")
    pluto.set_integrator(rk)
    try:
        pluto.load(w, ghost=ghost)
        dt0 = pluto.get_dt()
        pluto.step(4)
        ref = pluto.get_state()
        ref_dt, ref_t = pluto.get_dt(), pluto.get_time()
        pluto.load(w, ghost=ghost, nslab=nslab)
        assert pluto.get_dt() == dt0
        pluto.step(4)
        out = pluto.get_state()
        assert pluto.get_dt() == ref_dt and pluto.get_time() == ref_t
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])
    finally:
        pluto.set_integrator(2)


def test_slabs_against_the_oracle(pluto, oracle):
    """the decomposed step against the oracle directly (not only against the single-domain CUDA run)"""
    w = wl.random_smooth(40, 24, 21, seed=63, limiter=1)
    pluto.load(w, nslab=3)
    oracle.load(w)
    assert pluto.get_dt() == oracle.get_dt()
    pluto.step(2)
    assert oracle.step(2) == 0
    compare_state(pluto, oracle, w, TOL_1STEP_MAXREL)


def test_slab_argument_checks(pluto):
    from paper_2511_20337_b200 import binding
    with pytest.raises(binding.PlutoError):
        pluto.init(16, 16, 8, 2, nslab=4)            # 2 planes per slab < ghost + 1
    with pytest.raises(binding.PlutoError):
        pluto.init(16, 16, 1, 2, nslab=2)            # 2D box
    pluto.init(16, 16, 12, 2, nslab=4)
    k0, n = ctypes_int(), ctypes_int()
    assert pluto.L.pluto_local_planes(k0, n) == 0 and (k0.value, n.value) == (0, 12)


def ctypes_int():
    import ctypes
    return ctypes.c_int(0)


# ---------------------------------------------------------------- memory-safety checks of our own
# compute-sanitizer is closed on the GPU pool this repo is measured on, so the three properties its tools
# check are tested directly:
#   initcheck  -> a workspace poisoned with NaN bit patterns gives the same bits as a zeroed one
#   memcheck   -> guard bands around the registered workspace stay untouched
#   racecheck  -> repeated runs of every kernel variant give identical bits (a data race on shared or
#                 global memory between unsynchronised accesses shows up as run-to-run differences)

def _variant_cases():
    return [
        ("3d_wrap64_minmod", lambda: wl.random_smooth(64, 10, 9, seed=81, limiter=0), 2, 2, 1),
        ("3d_wrap128_mc", lambda: wl.random_smooth(128, 6, 5, seed=82, limiter=1), 2, 2, 1),
        ("3d_wrap96_rk3", lambda: wl.random_smooth(96, 7, 6, seed=89, limiter=0), 3, 2, 1),
        ("2d_wrap192", lambda: wl.random_smooth(192, 9, 1, seed=90, limiter=1), 2, 2, 1),
        ("3d_chunk_ragged", lambda: wl.random_smooth(37, 13, 11, seed=83, limiter=1), 3, 2, 1),
        ("3d_two_chunks", lambda: wl.random_smooth(300, 5, 4, seed=84, limiter=0), 2, 2, 1),
        ("2d_wrap64", lambda: wl.random_smooth(64, 20, 1, seed=85, limiter=1), 2, 2, 1),
        ("2d_chunk", lambda: wl.random_smooth(45, 17, 1, seed=86, limiter=0), 3, 2, 1),
        ("3d_wenoz", lambda: _wz(wl.random_smooth(40, 9, 8, seed=87)), 3, 3, 1),
        ("blast_24", lambda: wl.blast_3d(24), 2, 2, 1),
        ("3d_slabs", lambda: wl.random_smooth(64, 8, 12, seed=88, limiter=1), 2, 2, 3),
    ]


@pytest.mark.parametrize("name,make,rk,ghost,nslab", _variant_cases(), ids=[c[0] for c in _variant_cases()])
def test_poisoned_workspace_gives_the_same_bits(pluto, name, make, rk, ghost, nslab):
    """every byte of the device workspace is set to 0xFF (NaN patterns in every double) between pluto_init
    and pluto_set_state: a kernel that used a location the library had not written first would carry a
    NaN into the state"""
    w = make()
    pluto.set_integrator(rk)
    try:
        pluto.load(w, ghost=ghost, nslab=nslab)
        pluto.step(3)
        ref = pluto.get_state()
        ref_dt = pluto.get_dt()
        pluto.init(w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter, nslab=nslab)
        pluto.workspace.fill_(0xFF)
        pluto.torch.cuda.synchronize()
        pluto.set_box(*w.box)
        pluto.set_state(w.U, w.Bface)
        pluto.step(3)
        out = pluto.get_state()
        assert pluto.get_dt() == ref_dt
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])
    finally:
        pluto.set_integrator(2)


def test_guard_bands_around_the_workspace_stay_untouched(pluto):
    """the library computes inside the registered workspace only: 1 MiB of pattern on both sides of it is
    unchanged after every kernel variant has run"""
    import torch
    L = pluto.L
    guard = 1 << 20
    for name, make, rk, ghost, nslab in _variant_cases():
        w = make()
        need = L.pluto_workspace_bytes_slabs(nslab, 0, nslab, w.nx, w.ny, w.nz, ghost, rk)
        buf = torch.full((need + 2 * guard + 512,), 0xA5, dtype=torch.uint8, device=pluto.device)
        off = guard + (-(buf.data_ptr() + guard)) % 256
        torch.cuda.synchronize()
        assert L.pluto_finalize() == 0
        assert L.pluto_set_option(4, rk) >= 0
        assert L.pluto_set_workspace(buf.data_ptr() + off, need) == 0
        if nslab == 1:
            assert L.pluto_init(w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter) == 0
        else:
            assert L.pluto_init_slabs(nslab, 0, nslab, w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter) == 0
        assert L.pluto_set_box(*w.box) == 0
        assert L.pluto_set_state(w.U.ctypes.data, w.Bface.ctypes.data) == 0
        assert L.pluto_step(3) == 0 and L.pluto_step_fixed_dt(1, 1e-4) == 0
        U, B = np.empty_like(w.U), np.empty_like(w.Bface)
        assert L.pluto_get_state(U.ctypes.data, B.ctypes.data) == 0
        assert L.pluto_finalize() == 0
        torch.cuda.synchronize()
        assert bool((buf[:off] == 0xA5).all()) and bool((buf[off + need:] == 0xA5).all()), name
        assert np.isfinite(U).all()
    assert L.pluto_set_option(4, 2) >= 0
    pluto.workspace = None
    pluto.rk_order = 2


@pytest.mark.parametrize("name,make,rk,ghost,nslab", _variant_cases(), ids=[c[0] for c in _variant_cases()])
def test_repeated_runs_give_identical_bits(pluto, name, make, rk, ghost, nslab):
    """eight runs of five steps, CUDA-graph replay and plain launches alternating: identical bits every time"""
    from paper_2511_20337_b200.binding import OPT_GRAPH
    w = make()
    pluto.set_integrator(rk)
    try:
        ref = None
        for rep in range(8):
            pluto.set_option(OPT_GRAPH, rep & 1)
            pluto.load(w, ghost=ghost, nslab=nslab)
            pluto.step(5)
            out = pluto.get_state()
            if ref is None:
                ref = out
            assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1]), rep
    finally:
        pluto.set_option(OPT_GRAPH, 1)
        pluto.set_integrator(2)


# ---------------------------------------------------------------- GLM divergence cleaning (reading R20)

GLM_CASES = [
    ("2d_ragged_minmod", lambda: wl.random_smooth(37, 23, 1, seed=91, limiter=0, box=(1.0, 0.7, 1.0)), 2),
    ("2d_wide_mc_rk3", lambda: wl.random_smooth(150, 21, 1, seed=92, limiter=1), 3),
    ("3d_ragged_mc", lambda: wl.random_smooth(19, 13, 11, seed=93, limiter=1, box=(1.0, 0.8, 1.1)), 2),
    ("3d_minmod_rk3", lambda: wl.random_smooth(40, 12, 10, seed=94, limiter=0), 3),
    ("ot_48", lambda: wl.orszag_tang_2d(48), 2),
    ("blast_24", lambda: wl.blast_3d(24), 2),
]


def _glm_compare(pluto, oracle, tol, norm):
    Ug = pluto.get_state_glm()
    Uo, _ = oracle.get_state(faces=False)
    e_u = norm(Ug.reshape(8, -1), Uo.reshape(8, -1))
    pg, po = pluto.get_psi(), oracle.get_psi()
    e_p = norm(pg.reshape(1, -1), po.reshape(1, -1))
    assert e_u <= tol and e_p <= tol, (e_u, e_p)


@pytest.mark.parametrize("name,make,rk", GLM_CASES, ids=[c[0] for c in GLM_CASES])
def test_glm_parity(pluto, oracle, name, make, rk):
    """the GLM variant (cell-centred B + psi, [43]) against the oracle's: dt bit-exact, one step max-rel <= 1e-10,
    20 steps L1-rel <= 1e-8, strict per-component norms, psi included"""
    w = make()
    pluto.set_integrator(rk)
    try:
        pluto.load_glm(w)
        oracle.load_glm(w)
        oracle.set_integrator(rk)
        assert pluto.get_dt() == oracle.get_dt()
        pluto.step(1)
        assert oracle.step(1) == 0
        assert pluto.get_dt() == oracle.get_dt()
        _glm_compare(pluto, oracle, TOL_1STEP_MAXREL, maxrel)
        pluto.step(19)
        assert oracle.step(19) == 0
        _glm_compare(pluto, oracle, TOL_100STEP_L1REL, l1rel)
        assert abs(pluto.get_time() - oracle.get_time()) <= 1e-12
    finally:
        pluto.set_integrator(2)
        oracle.set_integrator(2)


def test_glm_conserves_and_cleans(pluto, oracle):
    """on the GPU itself: mass, momentum, energy and the cell-centred field are conserved; a divergence bump on a
    uniform magnetised fluid at rest is radiated away and damped (as in the oracle's pin)"""
    w = wl.random_smooth(32, 20, 12, seed=95, limiter=1)
    pluto.load_glm(w)
    pluto.step(30)
    U = pluto.get_state_glm()
    for v in range(8):
        ref = np.abs(w.U[1:4]).sum() if 1 <= v <= 3 else (np.abs(w.U[4:7]).sum() if 4 <= v <= 6 else abs(math.fsum(w.U[v].ravel())))
        assert abs(math.fsum(U[v].ravel()) - math.fsum(w.U[v].ravel())) <= 1e-12 * ref, v
    n = 64
    U0 = np.zeros((8, 1, n, n))
    X, Y = np.meshgrid((np.arange(n) + 0.5) / n, (np.arange(n) + 0.5) / n)
    U0[0] = 1.0
    U0[4, 0] = 0.3 + 1e-3 * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / 0.06 ** 2)
    U0[5, 0] = 0.2
    U0[7] = 1.0 / (5.0 / 3.0 - 1.0) + 0.5 * (U0[4] ** 2 + U0[5] ** 2)
    wb = wl.orszag_tang_2d(n)
    wb.U, wb.limiter, wb.cfl = U0, 1, 0.4

    def div(V):
        bx, by = V[4, 0], V[5, 0]
        return (np.roll(bx, -1, 1) - np.roll(bx, 1, 1)) * n / 2 + (np.roll(by, -1, 0) - np.roll(by, 1, 0)) * n / 2

    pluto.load_glm(wb)
    pluto.step(100)
    U1 = pluto.get_state_glm()
    assert math.sqrt((div(U1) ** 2).mean()) < 0.15 * math.sqrt((div(U0) ** 2).mean())
    psi = pluto.get_psi()
    pluto.set_psi(2.0 * psi)
    assert np.array_equal(pluto.get_psi(), 2.0 * psi)


def test_glm_argument_checks(pluto):
    from paper_2511_20337_b200 import binding
    pluto.set_divb(binding.DIVB_GLM)
    try:
        with pytest.raises(binding.PlutoError):
            pluto.init(16, 16, 16, 3, 5.0 / 3.0, 0.3, binding.WENOZ)       # PLM only
        with pytest.raises(binding.PlutoError):
            pluto.init(16, 16, 16, 2, nslab=2)                             # one domain
    finally:
        pluto.set_divb(binding.DIVB_CT)
    pluto.init(16, 16, 1, 2)
    with pytest.raises(binding.PlutoError):
        pluto.get_psi()                                                    # CT context has no psi


@pytest.mark.parametrize("rk", [2, 3])
def test_glm_poisoned_workspace_and_repeatability(pluto, rk):
    """the memory-safety checks of the CT path, for the GLM kernels: NaN-poisoned workspace, repeated runs"""
    from paper_2511_20337_b200 import binding
    w = wl.random_smooth(40, 13, 9, seed=96, limiter=1)
    pluto.set_integrator(rk)
    try:
        pluto.load_glm(w)
        pluto.step(4)
        ref, ref_psi = pluto.get_state_glm(), pluto.get_psi()
        for rep in range(3):
            pluto.set_divb(binding.DIVB_GLM)
            pluto.init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter)
            pluto.set_divb(binding.DIVB_CT)
            pluto.workspace.fill_(0xFF)
            pluto.torch.cuda.synchronize()
            pluto.set_box(*w.box)
            pluto._check(pluto.L.pluto_set_state(w.U.ctypes.data, None))
            pluto.step(4)
            assert np.array_equal(pluto.get_state_glm(), ref) and np.array_equal(pluto.get_psi(), ref_psi)
    finally:
        pluto.set_integrator(2)
