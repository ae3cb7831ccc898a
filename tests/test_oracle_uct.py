"""Pins for the UCT-HLLD EMF average of the oracle (reading R19; [47] named at PAPER.md:271, reference entry :640).
CPU only.  What is pinned, and by what:
  - the interface coefficients a^L, a^R, d^L, d^R and the transverse velocities: the composed 1D formula must
    equal the induction flux HLLD itself returns, in all six regions of the fan (the coefficients are the unique
    linear decomposition of that flux, so a wrong term anywhere fails this);
  - their mirror symmetry and their values for one-sided fans and for identical states;
  - the edge composition: equals the cell EMF on uniform data, equals -F_x[B_y] on y-invariant data, a grid-aligned
    run reproduces the 1D run along every axis (all three EMF components), div B and the conserved sums are kept,
    the Orszag-Tang point symmetry is kept, second order on the exact circularly polarised Alfven wave;
  - conditioning: a 1e-13 perturbation of the blast with its fluid at rest is not amplified (the weights are
    Lipschitz in the state when B_n != 0).
"""
import math

import numpy as np
import pytest

from paper_2511_20337_b200 import workloads as wl
from test_oracle_scheme import _embed, divb, ksum

G = 5.0 / 3.0


def _random_state(rng):
    return np.array([rng.uniform(0.1, 2), rng.normal() * rng.choice([0.1, 1, 3]), rng.normal(), rng.normal(),
                     rng.normal(), rng.normal(), rng.uniform(0.05, 2)])


def test_coefficients_reproduce_the_hlld_induction_flux(oracle):
    """F[B_t] = a^L (u B_t)^L + a^R (u B_t)^R - (d^R B_t^R - d^L B_t^L) - B_n (a^L v_t^L + a^R v_t^R)"""
    rng = np.random.default_rng(47)
    regions = {}
    for _ in range(6000):
        VL, VR = _random_state(rng), _random_state(rng)
        Bn = rng.normal() * rng.choice([0.0, 0.1, 1.0])
        F, u, dbg = oracle.hlld_uct(VL, VR, Bn, G)
        aL, dL, dR = u[0], u[1], u[2]
        aR = 1.0 - aL
        reg = int(dbg[6])
        regions[reg] = regions.get(reg, 0) + 1
        assert 0.0 <= aL <= 1.0
        for t, (ib, iF) in enumerate(((4, 5), (5, 6))):
            comp = aL * VL[1] * VL[ib] + aR * VR[1] * VR[ib] - (dR * VR[ib] - dL * VL[ib]) - Bn * u[3 + t]
            scale = max(1.0, abs(F[iF]), abs(VL[1] * VL[ib]), abs(VR[1] * VR[ib]))
            assert abs(comp - F[iF]) <= 1e-11 * scale, (reg, VL, VR, Bn)
        # the transverse velocities are the a-weighted means
        assert abs(u[3] - (aL * VL[2] + aR * VR[2])) <= 1e-15 * (1 + abs(u[3]))
        assert abs(u[4] - (aL * VL[3] + aR * VR[3])) <= 1e-15 * (1 + abs(u[4]))
    assert all(regions.get(r, 0) > 20 for r in range(6)), regions          # every region was sampled


def test_coefficients_special_cases(oracle):
    rng = np.random.default_rng(5)
    for _ in range(300):
        V = _random_state(rng)
        V[1] = rng.normal() * 0.3
        Bn = rng.normal()
        # identical states: d^L = d^R (the dissipative part cancels) and the flux is the physical one
        F, u, dbg = oracle.hlld_uct(V, V, Bn, G)
        if 0 < int(dbg[6]) < 5:
            assert abs(u[1] - u[2]) <= 1e-13 * (1 + abs(u[1]))
            assert u[1] >= -1e-14
        # mirror: swap sides, reverse the normal velocity and the normal field  =>  a^L <-> a^R, d^L <-> d^R
        VL, VR = _random_state(rng), _random_state(rng)
        _, u1, _ = oracle.hlld_uct(VL, VR, Bn, G)
        ML, MR = VR.copy(), VL.copy()
        ML[1] *= -1
        MR[1] *= -1
        _, u2, _ = oracle.hlld_uct(ML, MR, -Bn, G)
        assert abs(u1[0] - (1.0 - u2[0])) <= 1e-13
        assert abs(u1[1] - u2[2]) <= 1e-12 * (1 + abs(u1[1])) and abs(u1[2] - u2[1]) <= 1e-12 * (1 + abs(u1[2]))
    # one-sided fans: pure upwinding
    V = np.array([1.0, 5.0, 0.3, -0.2, 0.5, 0.1, 0.4])
    W = np.array([0.8, 4.0, 0.1, 0.2, 0.4, -0.3, 0.5])
    _, u, dbg = oracle.hlld_uct(V, W, 0.7, G)
    assert int(dbg[6]) == 0 and tuple(u[:3]) == (1.0, 0.0, 0.0) and u[3] == V[2] and u[4] == V[3]
    V[1] = W[1] = -5.0
    _, u, dbg = oracle.hlld_uct(V, W, 0.7, G)
    assert int(dbg[6]) == 5 and tuple(u[:3]) == (0.0, 0.0, 0.0) and u[3] == W[2] and u[4] == W[3]
    # fluid at rest, no field: both Alfven speeds vanish, nu* is taken as 0 (a^L = 1/2), everything finite
    V = np.array([1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0])
    _, u, _ = oracle.hlld_uct(V, V, 0.0, G)
    assert u[0] == 0.5 and np.all(np.isfinite(u))


def _load(oracle, w, rk=2):
    oracle.load(w)
    assert oracle.set_emf(1) == 0
    assert oracle.set_integrator(rk) == 0
    return oracle


def test_uniform_state_gives_the_cell_emf_and_is_a_fixed_point(oracle):
    nx, ny, nz = 5, 4, 6
    shp = (nz, ny, nx)
    v = np.array([0.4, -0.3, 0.2])
    B = np.array([0.5, 0.8, -0.6])
    U = wl.conserved_from_fields(np.full(shp, 1.1), [np.full(shp, x) for x in v], [np.full(shp, x) for x in B],
                                 np.full(shp, 0.9), G)
    Bf = wl.join_faces({nm: np.full(s, B["xyz".index(nm[1])]) for nm, s in wl.face_shapes(nx, ny, nz)}, nx, ny, nz)
    oracle.init(nx, ny, nz, 2, G, 0.3, 0)
    oracle.set_emf(1)
    oracle.set_state(U, Bf)
    E = oracle.debug_euler(0.01, want=("E",))["E"]
    Ec = -np.cross(v, B)
    for e in range(3):
        assert np.allclose(E[e], Ec[e], rtol=1e-13, atol=1e-14)
    assert oracle.step(3) == 0
    U1, Bf1 = oracle.get_state()
    assert np.abs(U1 - U).max() <= 1e-15 and np.array_equal(Bf1, Bf)
    oracle.set_emf(0)


def test_emf_reduces_to_1d_flux_for_invariant_data(oracle):
    """y-invariant data => Ez(i-1/2, j-1/2) = -F_x[B_y](i-1/2): the composition is the 1D formula"""
    w1 = wl.random_smooth(16, 1, 1, seed=5)
    nx, ny = 16, 6
    U = np.repeat(w1.U, ny, axis=2)
    f1 = wl.split_faces(w1.Bface, 16, 1, 1)
    By0 = w1.U[5, 0, 0, :]
    faces = {"bx": np.repeat(f1["bx"], ny, axis=1), "by": np.repeat(By0[None, None, :], ny + 1, axis=1)}
    oracle.init(nx, ny, 1, 2, G, 0.3, 0)
    oracle.set_emf(1)
    oracle.set_box(1.0, 1.0, 1.0)
    oracle.set_state(U, wl.join_faces(faces, nx, ny, 1))
    out = oracle.debug_euler(0.003, want=("E", "F"))
    Ez, Fx_By = out["E"][2], out["F"][0, 5]
    assert np.abs(Ez + Fx_By).max() <= 1e-13 * (1 + np.abs(Fx_By).max())
    assert np.abs(Fx_By).max() > 1e-3
    oracle.set_emf(0)


@pytest.mark.parametrize("limiter", [0, 1, 2])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_grid_aligned_run_reproduces_the_1d_solution(oracle, axis, limiter):
    """the discontinuous 1D problem of test_oracle_scheme, posed along every axis with UCT-HLLD: equals the 1D run
    (whose EMF rule does not matter: in 1D both reduce to the HLLD flux)"""
    n = 32
    x = wl.cell_centres(n, 1.0)
    left = (x > 0.25) & (x < 0.75)
    rho, p = np.where(left, 1.0, 0.125), np.where(left, 1.0, 0.1)
    vel = [0.2 * np.sin(2 * np.pi * x), 0.1 * np.cos(2 * np.pi * x), 0.05 * np.sin(4 * np.pi * x)]
    Bc = [np.full(n, 0.75), np.where(left, 1.0, -1.0), 0.3 * np.cos(2 * np.pi * x)]
    shp = (1, 1, n)
    U1 = wl.conserved_from_fields(rho.reshape(shp), [a.reshape(shp) for a in vel], [a.reshape(shp) for a in Bc],
                                  p.reshape(shp), 2.0)
    w1 = wl.Workload("bw", n, 1, 1, (1.0, 1.0, 1.0), 2.0, 0.3, limiter, 12, U1,
                     wl.join_faces({"bx": np.full((1, 1, n + 1), 0.75)}, n, 1, 1))
    oracle.load(w1)                                                   # 1D reference with the default rule
    dts = []
    for _ in range(12):
        assert oracle.step(1) == 0
        dts.append(oracle.get_dt())
    Uref, _ = oracle.get_state()
    shape, box, U, Bf, perm, along = _embed(w1, axis, 5)
    assert oracle.init(*shape, 2, 2.0, 0.3, limiter) == 0
    assert oracle.set_emf(1) == 0
    oracle.set_box(*box)
    oracle.set_state(U, Bf)
    for dt in dts:
        assert oracle.step_fixed_dt(1, dt) == 0
    Um, _ = oracle.get_state()
    comp = {0: 0, 7: 7}
    for m in range(3):
        comp[1 + m] = 1 + perm[m]
        comp[4 + m] = 4 + perm[m]
    for v in range(8):
        ref = along(Uref[v, 0, 0, :])
        assert np.abs(Um[comp[v]] - ref).max() <= 1e-12 * max(np.abs(ref).max(), 1.0), (v, axis)
    oracle.set_emf(0)


def test_conservation_divb_and_symmetry(oracle):
    w = wl.orszag_tang_2d(48, noise=0.0)
    _load(oracle, w)
    tot0 = [ksum(w.U[v]) for v in (0, 7)]
    assert oracle.step(40) == 0
    U, Bf = oracle.get_state()
    for n, v in enumerate((0, 7)):
        assert abs(ksum(U[v]) - tot0[n]) <= 1e-12 * abs(tot0[n])
    d = divb(Bf, w.nx, w.ny, w.nz, w.box)
    assert np.abs(d).max() * (w.box[0] / w.nx) <= 1e-12 * np.abs(Bf).max()
    flip = lambda a: a[:, ::-1, ::-1]
    for v, s in ((0, 1), (7, 1), (1, -1), (2, -1), (4, -1), (5, -1)):
        assert np.abs(U[v] - s * flip(U[v])).max() <= 1e-11 * np.abs(U[v]).max(), v
    # 3D, RK3
    w = wl.random_smooth(10, 9, 8, seed=3, box=(1.0, 0.8, 1.1))
    _load(oracle, w, rk=3)
    tot0 = [ksum(w.U[v]) for v in (0, 7)]
    assert oracle.step(10) == 0
    U, Bf = oracle.get_state()
    for n, v in enumerate((0, 7)):
        assert abs(ksum(U[v]) - tot0[n]) <= 1e-12 * abs(tot0[n])
    d = divb(Bf, w.nx, w.ny, w.nz, w.box)
    assert np.abs(d).max() * min(w.box[a] / n for a, n in enumerate((w.nx, w.ny, w.nz))) <= 1e-12 * np.abs(Bf).max()
    oracle.set_integrator(2)
    oracle.set_emf(0)


def _cpa_error(oracle, w, emf):
    oracle.load(w)
    oracle.set_emf(emf)
    t = 0.0
    while True:
        U, Bf = oracle.get_state()
        oracle.set_state(U, Bf)
        dt = oracle.get_dt()
        if t + dt < w.t_end:
            assert oracle.step_fixed_dt(1, dt) == 0
            t += dt
        else:
            assert oracle.step_fixed_dt(1, w.t_end - t) == 0
            break
    U, _ = oracle.get_state()
    oracle.set_emf(0)
    return math.sqrt(sum(np.abs(U[4 + s] - w.U[4 + s]).mean() ** 2 for s in range(3)))


def test_cp_alfven_3d_second_order(oracle):
    """the oblique wave of config 1 is genuinely three-dimensional for the EMF rule"""
    e16 = _cpa_error(oracle, wl.cp_alfven_3d(16, noise=0.0), 1)
    e32 = _cpa_error(oracle, wl.cp_alfven_3d(32, noise=0.0), 1)
    assert math.log2(e16 / e32) >= 1.7, (e16, e32)
    r32 = _cpa_error(oracle, wl.cp_alfven_3d(32, noise=0.0), 0)
    assert 0.5 * r32 <= e32 <= 1.5 * r32, (e32, r32)                 # same accuracy class as the default rule


def test_blast_at_rest_is_well_conditioned(oracle):
    """configs 3/4 start with the fluid at rest: a 1e-13 perturbation must not be amplified by the EMF rule"""
    w = wl.blast_3d(20)
    states = []
    for eps in (0.0, 1e-13):
        U = w.U.copy()
        rng = np.random.default_rng(9)
        fac = 1.0 + eps * rng.uniform(-1, 1, U[0].shape)
        U[0] *= fac
        oracle.init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter)
        oracle.set_box(*w.box)
        oracle.set_emf(1)
        oracle.set_state(U, w.Bface)
        assert oracle.step(8) == 0
        states.append(oracle.get_state())
    oracle.set_emf(0)
    for v in range(8):
        scale = np.abs(states[0][0][v]).max()
        if v in (1, 2, 3):
            scale = max(np.abs(states[0][0][a]).max() for a in (1, 2, 3))
        assert np.abs(states[0][0][v] - states[1][0][v]).max() <= 1e-10 * scale, v
    assert np.abs(states[0][1] - states[1][1]).max() <= 1e-10 * np.abs(states[0][1]).max()


def _rotate90(U, Bf, n):
    """the 2D state on an n x n periodic unit square rotated by +90 degrees: point (x, y) -> (1 - y, x), vectors
    (a_x, a_y) -> (-a_y, a_x); cell (i, j) -> (n - 1 - j, i), y-face (i, j - 1/2) -> x-face (n - j, i) with
    b_x' = -b_y, x-face (i - 1/2, j) -> y-face (n - 1 - j, i) with b_y' = b_x"""
    f = wl.split_faces(Bf, n, n, 1)
    Ur = np.empty_like(U)
    rot = lambda a: np.ascontiguousarray(a[0].T[:, ::-1])[None]           # q'[j' = i][i' = n-1-j] = q[j][i]
    for v in (0, 3, 6, 7):
        Ur[v] = rot(U[v])
    Ur[1], Ur[2] = -rot(U[2]), rot(U[1])
    Ur[4], Ur[5] = -rot(U[5]), rot(U[4])
    bx, by = f["bx"][0], f["by"][0]                                      # [n][n+1], [n+1][n]
    bxr = np.empty_like(bx)
    byr = np.empty_like(by)
    for j in range(n + 1):
        bxr[:, n - j] = -by[j, :]                                         # bx'[j' = i][n - j] = -by[j][i]
    for j in range(n):
        byr[:, n - 1 - j] = bx[j, :]                                      # by'[j'_f = i][i' = n-1-j] = bx[j][i]
    return Ur, wl.join_faces({"bx": bxr[None], "by": byr[None]}, n, n, 1)


@pytest.mark.parametrize("emf", [0, 1])
def test_quarter_turn_covariance(oracle, emf):
    """the scheme commutes with a rotation of the square grid by 90 degrees: the orientation and the signs of the
    two-dimensional edge composition (both rules) are consistent between the x and the y direction"""
    n = 24
    w = wl.random_smooth(n, n, 1, seed=31, limiter=1, amp=0.3, box=(1.0, 1.0, 1.0))
    oracle.load(w)
    oracle.set_emf(emf)
    dts = []
    for _ in range(6):
        assert oracle.step(1) == 0
        dts.append(oracle.get_dt())
    Ua, Ba = oracle.get_state()
    Ur0, Br0 = _rotate90(w.U, w.Bface, n)
    assert oracle.init(n, n, 1, 2, w.gamma, w.cfl, 1) == 0
    oracle.set_emf(emf)
    oracle.set_box(1.0, 1.0, 1.0)
    oracle.set_state(Ur0, Br0)
    for dt in dts:
        assert oracle.step_fixed_dt(1, dt) == 0
    Ub, Bb = oracle.get_state()
    oracle.set_emf(0)
    Ue, Be = _rotate90(Ua, Ba, n)
    assert np.abs(Ub - Ue).max() <= 1e-12 * np.abs(Ue).max()
    assert np.abs(Bb - Be).max() <= 1e-12 * np.abs(Be).max()
    assert np.abs(Ua - w.U).max() > 1e-3                                  # something happened


@pytest.mark.parametrize("emf", [0, 1])
def test_cyclic_permutation_of_the_axes_3d(oracle, emf):
    """a genuinely 3D state with the axes renamed cyclically (new x = old y, new y = old z, new z = old x) advances
    to the renamed result: all three EMF components are one formula under the cyclic map (both rules)"""
    w = wl.random_smooth(10, 8, 6, seed=41, limiter=1, amp=0.3, box=(1.0, 0.8, 0.6))
    oracle.load(w)
    oracle.set_emf(emf)
    dts = []
    for _ in range(4):
        assert oracle.step(1) == 0
        dts.append(oracle.get_dt())
    Ua, Ba = oracle.get_state()

    def rename(U, Bf):
        f = wl.split_faces(Bf, w.nx, w.ny, w.nz)
        tr = lambda a: np.ascontiguousarray(np.transpose(a, (2, 0, 1)))       # q'[i][k][j] = q[k][j][i]
        Ur = np.empty((8, w.nx, w.nz, w.ny))
        Ur[0], Ur[7] = tr(U[0]), tr(U[7])
        for base in (1, 4):                                                    # a'_x = a_y, a'_y = a_z, a'_z = a_x
            Ur[base + 0], Ur[base + 1], Ur[base + 2] = tr(U[base + 1]), tr(U[base + 2]), tr(U[base + 0])
        faces = {"bx": tr(f["by"]), "by": tr(f["bz"]), "bz": tr(f["bx"])}
        return Ur, wl.join_faces(faces, w.ny, w.nz, w.nx)
    Ur0, Br0 = rename(w.U, w.Bface)
    assert oracle.init(w.ny, w.nz, w.nx, 2, w.gamma, w.cfl, 1) == 0
    oracle.set_emf(emf)
    oracle.set_box(w.box[1], w.box[2], w.box[0])
    oracle.set_state(Ur0, Br0)
    for dt in dts:
        assert oracle.step_fixed_dt(1, dt) == 0
    Ub, Bb = oracle.get_state()
    oracle.set_emf(0)
    Ue, Be = rename(Ua, Ba)
    assert np.abs(Ub - Ue).max() <= 1e-12 * np.abs(Ue).max()
    assert np.abs(Bb - Be).max() <= 1e-12 * np.abs(Be).max()
    assert np.abs(Ua - w.U).max() > 1e-3
