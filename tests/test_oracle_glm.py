"""Pins of the oracle's GLM divergence-cleaning variant (reading R20; [43] PAPER.md:636):
the exact (B_n, psi) interface state against the jump conditions of its two waves, the reduction to the
CT scheme in 1D, conservation (now including the cell-centred field), the exact damping of psi, the
transport of a divergence error at +-c_h, the decay of a 2D divergence error, second-order convergence on
the exact circularly polarised Alfven wave."""
import math

import numpy as np
import pytest

from paper_2511_20337_b200 import workloads as wl


def test_interface_state_satisfies_both_jump_conditions(oracle):
    """the subsystem dB/dt + dpsi/dx = 0, dpsi/dt + ch^2 dB/dx = 0 has flux f(B, psi) = (psi, ch^2 B); across the
    wave of speed s the Rankine-Hugoniot condition is f_b - f_a = s (U_b - U_a): -ch between the left and the
    middle state, +ch between the middle and the right state"""
    rng = np.random.default_rng(3)
    for _ in range(200):
        BL, BR, pL, pR = rng.normal(size=4)
        ch = float(rng.uniform(0.3, 5.0))
        Bm, pm = oracle.glm_interface(BL, BR, pL, pR, ch)
        # wave -ch: (left, middle)
        assert abs((pm - pL) - (-ch) * (Bm - BL)) <= 1e-13 * (1 + ch)
        assert abs(ch * ch * (Bm - BL) - (-ch) * (pm - pL)) <= 1e-13 * (1 + ch) ** 2
        # wave +ch: (middle, right)
        assert abs((pR - pm) - ch * (BR - Bm)) <= 1e-13 * (1 + ch)
        assert abs(ch * ch * (BR - Bm) - ch * (pR - pm)) <= 1e-13 * (1 + ch) ** 2
    assert oracle.glm_interface(0.7, 0.7, -0.2, -0.2, 2.0) == (0.7, -0.2)      # consistency


def test_1d_run_equals_the_constrained_transport_run(oracle):
    """in 1D the normal field is constant: B_m = B_x, psi stays zero, and the GLM variant IS the base scheme"""
    w = wl.cp_alfven_1d(64)
    oracle.load(w)
    dts = []
    for _ in range(20):
        oracle.step(1)
        dts.append(oracle.get_dt())
    Uc, _ = oracle.get_state()
    oracle.load_glm(w)
    for dt in dts:
        assert oracle.step(1) == 0 and oracle.get_dt() == dt
    Ug, _ = oracle.get_state(faces=False)
    assert np.abs(Ug - Uc).max() <= 1e-14
    assert np.abs(oracle.get_psi()).max() == 0.0


@pytest.mark.parametrize("shape,rk", [((24, 16, 1), 2), ((12, 10, 8), 3)])
def test_conservation_including_the_field(oracle, shape, rk):
    w = wl.random_smooth(*shape, seed=7, limiter=1)
    oracle.load_glm(w)
    oracle.set_integrator(rk)
    tot0 = [math.fsum(w.U[v].ravel()) for v in range(8)]
    assert oracle.step(30) == 0
    U, _ = oracle.get_state(faces=False)
    scale = {1: np.abs(w.U[1:4]).sum(), 2: np.abs(w.U[1:4]).sum(), 3: np.abs(w.U[1:4]).sum(),
             4: np.abs(w.U[4:7]).sum(), 5: np.abs(w.U[4:7]).sum(), 6: np.abs(w.U[4:7]).sum()}
    for v in range(8):
        ref = scale.get(v, abs(tot0[v]))
        assert abs(math.fsum(U[v].ravel()) - tot0[v]) <= 1e-12 * ref, v
    oracle.set_integrator(2)


def test_uniform_psi_decays_exactly(oracle):
    """uniform state, uniform psi: every flux difference vanishes and psi(t + dt) = psi exp(-dt ch / 0.18),
    ch = cfl min(dx) / dt"""
    w = wl.random_smooth(8, 6, 4, seed=1, amp=0.0)
    oracle.load_glm(w)
    psi0 = 0.37
    oracle.set_psi(np.full((w.nz, w.ny, w.nx), psi0))
    U0, _ = oracle.get_state(faces=False)
    dt = oracle.get_dt()
    assert oracle.step(1) == 0
    ch = w.cfl * min(w.box[0] / w.nx, w.box[1] / w.ny, w.box[2] / w.nz) / dt
    assert np.abs(oracle.get_psi() - psi0 * math.exp(-dt * ch / 0.18)).max() <= 1e-15
    U1, _ = oracle.get_state(faces=False)
    assert np.array_equal(U0, U1)


def test_divergence_error_travels_at_ch(oracle):
    """a tiny bump of the normal field on a fluid at rest splits into two pulses moving at -ch and +ch"""
    n = 256
    U = np.zeros((8, 1, 1, n))
    x = (np.arange(n) + 0.5) / n
    U[0] = 1.0
    bump = 1e-8 * np.exp(-((x - 0.5) / 0.03) ** 2)
    U[4, 0, 0] = 0.5 + bump
    U[7] = 1.0 / (5.0 / 3.0 - 1.0) + 0.5 * U[4] ** 2
    assert oracle.init(n, 1, 1, 2, 5.0 / 3.0, 0.4, 1) == 0
    assert oracle.set_box(1.0, 1.0, 1.0) == 0 and oracle.set_divb(1) == 0
    assert oracle.set_state(U, None) == 0
    t = 0.0
    for _ in range(40):
        assert oracle.step(1) == 0
    t = oracle.get_time()
    dt = oracle.get_dt()
    ch = 0.4 * (1.0 / n) / dt
    Ug, _ = oracle.get_state(faces=False)
    d = Ug[4, 0, 0] - 0.5
    right, left = d[n // 2:], d[:n // 2]
    xr = (x[n // 2:] * right).sum() / right.sum()
    xl = (x[:n // 2] * left).sum() / left.sum()
    # dt (hence ch) is constant here: the fluid stays at rest to O(1e-16)
    assert abs(xr - (0.5 + ch * t)) <= 2.0 / n and abs(xl - (0.5 - ch * t)) <= 2.0 / n
    assert abs(right.sum() - left.sum()) <= 1e-3 * abs(right.sum())


def test_divergence_error_is_cleaned_in_2d(oracle):
    """a monopole-like bump of B_x on a uniform magnetised fluid at rest: the cleaning radiates the divergence
    away at c_h and damps it (rms of the central-difference divergence: 27 % after 50 steps, 9 % after 100)"""
    n = 64
    U = np.zeros((8, 1, n, n))
    X, Y = np.meshgrid((np.arange(n) + 0.5) / n, (np.arange(n) + 0.5) / n)
    U[0] = 1.0
    U[4, 0] = 0.3 + 1e-3 * np.exp(-((X - 0.5) ** 2 + (Y - 0.5) ** 2) / 0.06 ** 2)
    U[5, 0] = 0.2
    U[7] = 1.0 / (5.0 / 3.0 - 1.0) + 0.5 * (U[4] ** 2 + U[5] ** 2)

    def div(V):
        bx, by = V[4, 0], V[5, 0]
        return (np.roll(bx, -1, 1) - np.roll(bx, 1, 1)) * n / 2 + (np.roll(by, -1, 0) - np.roll(by, 1, 0)) * n / 2

    assert oracle.init(n, n, 1, 2, 5.0 / 3.0, 0.4, 1) == 0
    assert oracle.set_box(1.0, 1.0, 1.0) == 0 and oracle.set_divb(1) == 0
    assert oracle.set_state(U, None) == 0
    d0 = math.sqrt((div(U) ** 2).mean())
    assert oracle.step(100) == 0
    U1, _ = oracle.get_state(faces=False)
    d1 = math.sqrt((div(U1) ** 2).mean())
    assert d1 < 0.15 * d0 and np.abs(div(U1)).max() < 0.05 * np.abs(div(U)).max(), (d0, d1)
    assert 0.0 < np.abs(oracle.get_psi()).max() < 1e-3


def test_cp_alfven_3d_second_order(oracle):
    """the exact oblique circularly polarised Alfven wave (Eq. 10; configs[1] without noise),
    one period: the cell-centred GLM variant converges at second order like the CT scheme"""
    errs = []
    for n in (16, 32):
        w = wl.cp_alfven_3d(n, noise=0.0)
        oracle.load_glm(w)
        t = 0.0
        while True:
            U, _ = oracle.get_state(faces=False)
            psi = oracle.get_psi()
            oracle.set_state(U, None)
            oracle.set_psi(psi)
            dt = oracle.get_dt()
            if t + dt < w.t_end:
                assert oracle.step_fixed_dt(1, dt) == 0
                t += dt
            else:
                assert oracle.step_fixed_dt(1, w.t_end - t) == 0
                break
        U, _ = oracle.get_state(faces=False)
        errs.append(math.sqrt(sum(np.abs(U[4 + s] - w.U[4 + s]).mean() ** 2 for s in range(3))))
    order = math.log2(errs[0] / errs[1])
    assert order >= 1.5, (errs, order)
