"""Pins for the pieces of the oracle (CPU only).  Each test checks oracle/oracle.c against something
other than itself: a closed form, a textbook special case, a symmetry or a jump condition, chosen so
that a dropped term, a wrong sign or a transposed operand fails one of them (SURVEY 8(c) pin table)."""
import math

import numpy as np
import pytest

G = 5.0 / 3.0
rng = np.random.default_rng(12345)


def rand_state(r=rng, B=True):
    """rotated-frame primitive state (rho,u,v,w,By,Bz,p)"""
    V = np.array([r.uniform(0.2, 3), r.uniform(-1.5, 1.5), r.uniform(-1, 1), r.uniform(-1, 1),
                  r.uniform(-1.5, 1.5), r.uniform(-1.5, 1.5), r.uniform(0.1, 3)])
    if not B:
        V[4] = V[5] = 0.0
    return V


# ------------------------------------------------------------------ cons <-> prim (Eq. 3, Eq. 7)

def test_cons2prim_closed_form_and_roundtrip(oracle):
    for _ in range(200):
        V = np.array([rng.uniform(0.1, 5), *rng.uniform(-2, 2, 3), *rng.uniform(-2, 2, 3), rng.uniform(0.05, 5)])
        U = oracle.prim2cons(V, G)
        # closed form written independently (Eq. 3)
        E = V[7] / (G - 1) + 0.5 * V[0] * np.dot(V[1:4], V[1:4]) + 0.5 * np.dot(V[4:7], V[4:7])
        assert U[0] == V[0] and np.allclose(U[1:4], V[0] * V[1:4], rtol=1e-15) and np.all(U[4:7] == V[4:7])
        assert abs(U[7] - E) <= 4e-16 * abs(E)
        rc, V2 = oracle.cons2prim(U, G)
        assert rc == 0
        assert np.allclose(V2, V, rtol=2e-14, atol=2e-14)


def test_cons2prim_flags_unphysical(oracle):
    rc, _ = oracle.cons2prim(np.array([1.0, 0, 0, 0, 0, 0, 0, -1.0]), G)
    assert rc != 0
    rc, _ = oracle.cons2prim(np.array([-1.0, 0, 0, 0, 0, 0, 0, 1.0]), G)
    assert rc != 0
    rc, _ = oracle.cons2prim(np.array([1.0, 0, 0, 0, 0, 0, 0, np.nan]), G)
    assert rc != 0


# ------------------------------------------------------------------ fast speed

def test_fast_speed_special_cases(oracle):
    for _ in range(100):
        rho, p = rng.uniform(0.1, 4), rng.uniform(0.1, 4)
        a = np.sqrt(G * p / rho)
        # B = 0 -> sound speed
        assert abs(oracle.fast_speed(rho, p, 0, 0, 0, G) - a) < 1e-14 * a
        # field along the normal only -> max(a, Alfven)
        Bn = rng.uniform(-3, 3)
        ca = abs(Bn) / np.sqrt(rho)
        assert abs(oracle.fast_speed(rho, p, Bn, 0, 0, G) - max(a, ca)) < 1e-7 * max(a, ca)
        # field perpendicular to the normal -> sqrt(a^2 + b^2)
        Bt1, Bt2 = rng.uniform(-2, 2, 2)
        ref = np.sqrt(a * a + (Bt1 ** 2 + Bt2 ** 2) / rho)
        assert abs(oracle.fast_speed(rho, p, 0.0, Bt1, Bt2, G) - ref) < 1e-14 * ref
        # general: root of the magnetosonic quartic c^4 - (a^2+b^2) c^2 + a^2 bn^2 = 0, the larger one
        cf = oracle.fast_speed(rho, p, Bn, Bt1, Bt2, G)
        b2 = (Bn ** 2 + Bt1 ** 2 + Bt2 ** 2) / rho
        assert abs(cf ** 4 - (a * a + b2) * cf ** 2 + a * a * Bn ** 2 / rho) < 1e-12 * cf ** 4
        assert cf * cf >= 0.5 * (a * a + b2) - 1e-14


# ------------------------------------------------------------------ PLM (R4)

@pytest.mark.parametrize("lim", [0, 1])
def test_plm_linear_data_and_extrema(oracle, lim):
    for _ in range(100):
        s = rng.uniform(-3, 3)
        assert oracle.plm_slope(s, s, lim) == s                   # linear data reproduced exactly
        a, b = rng.uniform(0.1, 3, 2)
        assert oracle.plm_slope(a, -b, lim) == 0.0                # extremum -> zero slope
        assert oracle.plm_slope(-a, b, lim) == 0.0
        assert oracle.plm_slope(0.0, b, lim) == 0.0
        # antisymmetry and symmetry in the arguments
        assert oracle.plm_slope(-a, -b, lim) == -oracle.plm_slope(a, b, lim)
        assert oracle.plm_slope(a, b, lim) == oracle.plm_slope(b, a, lim)


def test_minmod_and_mc_values(oracle):
    for _ in range(200):
        a, b = rng.uniform(0.01, 3, 2)
        assert oracle.plm_slope(a, b, 0) == min(a, b)
        mc = oracle.plm_slope(a, b, 1)
        assert mc == min(2 * a, 2 * b, 0.5 * (a + b))
        if 1.0 / 3.0 <= a / b <= 3.0:
            assert mc == 0.5 * (a + b)                            # central slope inside [1/3, 3]
        assert oracle.plm_slope(a, b, 0) <= mc <= 2 * min(a, b)    # TVD region


# ------------------------------------------------------------------ physical flux (Eq. 2)

def test_physical_flux_against_tensor_form(oracle):
    """T of Eq. 2 written with 3-vectors and contracted with e_x"""
    for _ in range(100):
        V = rand_state()
        Bn = rng.uniform(-1, 1)
        rho, vel, B, p = V[0], V[1:4], np.array([Bn, V[4], V[5]]), V[6]
        pt = p + 0.5 * B @ B
        E = p / (G - 1) + 0.5 * rho * vel @ vel + 0.5 * B @ B
        T_m = rho * np.outer(vel, vel) - np.outer(B, B) + pt * np.eye(3)
        T_B = np.outer(vel, B) - np.outer(B, vel)
        ref = np.concatenate([[rho * vel[0]], T_m[0], T_B[0], [(E + pt) * vel[0] - (vel @ B) * B[0]]])
        F = oracle.physical_flux(V, Bn, G)
        assert np.allclose(F, ref, rtol=1e-13, atol=1e-13)
        assert F[4] == 0.0


# ------------------------------------------------------------------ HLLD (R5)

def test_hlld_consistency(oracle):
    for _ in range(300):
        V = rand_state()
        Bn = rng.uniform(-1.5, 1.5)
        F, w = oracle.hlld(V, V, Bn, G)
        ref = oracle.physical_flux(V, Bn, G)
        assert np.allclose(F, ref, rtol=2e-13, atol=2e-13)


def test_hlld_mirror_symmetry(oracle):
    sgn = np.array([-1, 1, -1, -1, 1, -1, -1, -1.0])
    worst = 0.0
    for _ in range(3000):
        VL, VR = rand_state(), rand_state()
        Bn = rng.uniform(-1.5, 1.5)
        F, w = oracle.hlld(VL, VR, Bn, G)
        mL, mR = VR.copy(), VL.copy()
        mL[1] *= -1
        mR[1] *= -1
        Fm, wm = oracle.hlld(mL, mR, -Bn, G)
        scale = np.abs(F).max() + 1.0
        worst = max(worst, np.abs(Fm - sgn * F).max() / scale)
        assert abs((1.0 - wm) - w) < 1e-9
    assert worst < 1e-12


def _hllc_euler(VL, VR, SL, SR, g=G):
    """textbook HLLC (Toro) for the Euler equations with given outer speeds; V = (rho,u,v,w,p)"""
    def cons(V):
        rho, u, v, w, p = V
        return np.array([rho, rho * u, rho * v, rho * w, p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)])

    def flux(V):
        rho, u, v, w, p = V
        E = cons(V)[4]
        return np.array([rho * u, rho * u * u + p, rho * u * v, rho * u * w, (E + p) * u])
    rL, uL, pL = VL[0], VL[1], VL[4]
    rR, uR, pR = VR[0], VR[1], VR[4]
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))
    if SL >= 0:
        return flux(VL)
    if SR <= 0:
        return flux(VR)

    def star(V, S):
        rho, u, v, w, p = V
        E = cons(V)[4]
        f = rho * (S - u) / (S - Ss)
        return f * np.array([1, Ss, v, w, E / rho + (Ss - u) * (Ss + p / (rho * (S - u)))])
    if Ss >= 0:
        return flux(VL) + SL * (star(VL, SL) - cons(VL))
    return flux(VR) + SR * (star(VR, SR) - cons(VR))


def test_hlld_reduces_to_hllc_without_field(oracle):
    for _ in range(500):
        VL, VR = rand_state(B=False), rand_state(B=False)
        F, w, dbg = oracle.hlld(VL, VR, 0.0, G, debug=True)
        ref = _hllc_euler(VL[[0, 1, 2, 3, 6]], VR[[0, 1, 2, 3, 6]], dbg[0], dbg[1])
        assert np.all(np.isfinite(F))
        assert np.allclose(F[[0, 1, 2, 3, 7]], ref, rtol=1e-12, atol=1e-12)
        assert np.all(F[4:7] == 0.0)
        # outer speeds are min/max(u) -/+ max(sound speed)  (R5)
        cL, cR = np.sqrt(G * VL[6] / VL[0]), np.sqrt(G * VR[6] / VR[0])
        assert abs(dbg[0] - (min(VL[1], VR[1]) - max(cL, cR))) < 1e-13
        assert abs(dbg[1] - (max(VL[1], VR[1]) + max(cL, cR))) < 1e-13


def test_hlld_stationary_contact_is_exact(oracle):
    for _ in range(100):
        VL = rand_state()
        VL[1] = 0.0
        VR = VL.copy()
        VR[0] = rng.uniform(0.2, 3)          # jump in density only
        Bn = rng.uniform(-1, 1)
        F, w = oracle.hlld(VL, VR, Bn, G)
        v, ww, By, Bz, p = VL[2], VL[3], VL[4], VL[5], VL[6]
        pT = p + 0.5 * (Bn * Bn + By * By + Bz * Bz)
        vB = v * By + ww * Bz
        ref = np.array([0, pT - Bn * Bn, -Bn * By, -Bn * Bz, 0, -Bn * v, -Bn * ww, -Bn * vB])
        assert np.allclose(F, ref, rtol=1e-12, atol=1e-12)
        assert abs(F[0]) < 1e-13                                  # zero mass flux
        assert abs(w - 0.5) < 1e-6


def test_hlld_rankine_hugoniot_across_all_five_waves(oracle):
    """S (U_b - U_a) = F_b - F_a across S_L, S*_L, S_M, S*_R, S_R with the intermediate fluxes
    F*_a = F_a + S_a (U*_a - U_a), F**_a = F*_a + S*_a (U**_a - U*_a)   ([56] PAPER.md:649)"""
    n_checked = 0
    for _ in range(2000):
        VL, VR = rand_state(), rand_state()
        Bn = rng.uniform(-1.5, 1.5)
        if abs(Bn) < 0.05:
            continue
        F, w, d = oracle.hlld(VL, VR, Bn, G, debug=True)
        if d[6] in (0, 5):
            continue
        SL, SR, SM, pTs, SaL, SaR = d[0:6]
        UL, UR, UsL, UsR, UssL, UssR, FL, FR = (d[8 + 8 * m: 16 + 8 * m] for m in range(8))
        FsL = FL + SL * (UsL - UL)
        FsR = FR + SR * (UsR - UR)
        FssL = FsL + SaL * (UssL - UsL)
        FssR = FsR + SaR * (UssR - UsR)
        scale = max(np.abs(FL).max(), np.abs(FR).max(), 1.0)
        # contact: S_M (U**R - U**L) = F**R - F**L  (not imposed by construction: a real check)
        assert np.abs(SM * (UssR - UssL) - (FssR - FssL)).max() < 2e-11 * scale
        # star fluxes must be the physical flux form evaluated with (S_M, pT*):
        for Us, Fs in ((UsL, FsL), (UsR, FsR), (UssL, FssL), (UssR, FssR)):
            rho, mx, my, mz, Bx, By, Bz, E = Us
            u, v, ww = mx / rho, my / rho, mz / rho
            assert abs(u - SM) < 1e-12 * (1 + abs(SM))
            phys = np.array([rho * u, rho * u * u + pTs - Bx * Bx, rho * u * v - Bx * By, rho * u * ww - Bx * Bz,
                             0.0, By * u - Bx * v, Bz * u - Bx * ww,
                             (E + pTs) * u - Bx * (u * Bx + v * By + ww * Bz)])
            assert np.abs(phys - Fs).max() < 5e-11 * scale * (1 + np.abs(Us).max())
        # region selection (R5 order)
        reg = 1 if SaL >= 0 else 2 if SM >= 0 else 3 if SaR > 0 else 4
        assert d[6] == reg
        Fsel = (FsL, FssL, FssR, FsR)[reg - 1].copy()
        Fsel[4] = 0
        assert np.allclose(F, Fsel, rtol=1e-11, atol=1e-11 * scale)
        # Alfven speeds
        assert abs(SaL - (SM - abs(Bn) / np.sqrt(UsL[0]))) < 1e-13 * (1 + abs(SaL))
        assert abs(SaR - (SM + abs(Bn) / np.sqrt(UsR[0]))) < 1e-13 * (1 + abs(SaR))
        n_checked += 1
    assert n_checked > 1000


def test_hlld_supersonic_returns_upwind_flux(oracle):
    V = np.array([1.0, 10.0, 0.3, -0.2, 0.5, 0.1, 1.0])
    V2 = np.array([0.8, 9.0, 0.1, 0.2, 0.3, -0.1, 1.2])
    F, w = oracle.hlld(V, V2, 0.7, G)
    assert np.array_equal(F, oracle.physical_flux(V, 0.7, G))
    assert w == 1.0
    V[1] *= -1
    V2[1] *= -1
    F, w = oracle.hlld(V, V2, 0.7, G)
    assert np.array_equal(F, oracle.physical_flux(V2, 0.7, G))
    assert w == 0.0


def test_hlld_finite_in_degenerate_field_configurations(oracle):
    for _ in range(300):
        VL, VR = rand_state(), rand_state()
        F, w = oracle.hlld(VL, VR, 0.0, G)                         # Bx = 0, B_t != 0
        assert np.all(np.isfinite(F)) and 0.0 <= w <= 1.0
        VL[4:6] = 0
        VR[4:6] = 0
        F, w = oracle.hlld(VL, VR, rng.uniform(-1, 1), G)            # B along the normal only
        assert np.all(np.isfinite(F))
        # then the transverse field flux vanishes only if v_t = 0; check the hydro part is HLLC-like finite
    # switch-on degeneracy: D -> 0 when S_M = u and rho (S-u)^2 = Bx^2; build it on purpose
    rho, p = 1.0, 0.6
    Bn = np.sqrt(G * p) * 1.0000000001                                 # Alfven speed ~ sound speed
    V = np.array([rho, 0.0, 0.0, 0.0, 1e-9, 0.0, p])
    F, w = oracle.hlld(V, V, Bn, G)
    assert np.all(np.isfinite(F))


def test_upwind_weight_definition(oracle):
    """R6: w = clamp(1/2 + F_rho / (2 theta f_ref)), f_ref = (rho_L+rho_R)(S_R-S_L)/4, theta = 1e-3"""
    seen_mid = 0
    for _ in range(2000):
        VL, VR = rand_state(), rand_state()
        VL[1] *= 1e-4
        VR[1] = VL[1] + rng.uniform(-1, 1) * 1e-4
        VR[6] = VL[6] * (1 + 1e-4 * rng.uniform(-1, 1))
        VR[4:6] = VL[4:6]
        Bn = rng.uniform(-1, 1)
        F, w, d = oracle.hlld(VL, VR, Bn, G, debug=True)
        fref = 0.25 * (VL[0] + VR[0]) * (d[1] - d[0])
        ref = min(1.0, max(0.0, 0.5 + 0.5 * F[0] / (1e-3 * fref)))
        assert abs(w - ref) < 1e-12
        seen_mid += 0.0 < w < 1.0
    assert seen_mid > 100


# --------------------------------------------------------------------------- WENO-Z reconstruction ([51], R18)

def _wenoz(oracle, v):
    import ctypes
    v = np.ascontiguousarray(v, dtype=np.float64)
    return oracle.L.oracle_wenoz(v.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))


def test_wenoz_is_exact_for_quadratic_cell_averages(oracle):
    """every candidate stencil reproduces a parabola's face value from its cell averages, so any convex
    combination does: value at x = 1/2 of a + b x + c x^2 with averages a + b i + c (i^2 + 1/12)"""
    rng = np.random.default_rng(5)
    for _ in range(50):
        a, b, c = rng.normal(size=3)
        avg = [a + b * i + c * (i * i + 1.0 / 12.0) for i in range(-2, 3)]
        exact = a + 0.5 * b + 0.25 * c
        assert abs(_wenoz(oracle, avg) - exact) <= 1e-13 * (abs(a) + abs(b) + abs(c))


def test_wenoz_is_fifth_order_on_smooth_data(oracle):
    errs = []
    for h in (0.1, 0.05, 0.025):
        av = [(-math.cos(1 + (i + 0.5) * h) + math.cos(1 + (i - 0.5) * h)) / h for i in range(-2, 3)]
        errs.append(abs(_wenoz(oracle, av) - math.sin(1 + 0.5 * h)))
    assert math.log2(errs[0] / errs[1]) > 4.7 and math.log2(errs[1] / errs[2]) > 4.7


def test_wenoz_takes_the_smooth_side_of_a_jump_and_stays_bounded(oracle):
    assert abs(_wenoz(oracle, [0, 0, 0, 1, 1])) < 1e-30          # jump right of the face: left stencil only
    assert abs(_wenoz(oracle, [0, 0, 1, 1, 1]) - 1.0) < 1e-30    # jump left of the cell
    rng = np.random.default_rng(6)
    for _ in range(200):
        lo, hi = sorted(rng.normal(size=2))
        k = rng.integers(1, 5)
        v = [lo] * k + [hi] * (5 - k)
        r = _wenoz(oracle, v)
        assert lo - 1e-12 <= r <= hi + 1e-12
    assert _wenoz(oracle, [2.5] * 5) == pytest.approx(2.5, abs=1e-15)
    # mirror: the lower-face value of the mirrored data
    v = rng.normal(size=5)
    assert _wenoz(oracle, v[::-1]) != _wenoz(oracle, v)
    assert _wenoz(oracle, -v) == pytest.approx(-_wenoz(oracle, v), rel=1e-14)
