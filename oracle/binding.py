"""ctypes binding of liboracle.so (TEST INFRASTRUCTURE ONLY; see oracle/oracle.h)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "oracle.c"), os.path.join(_HERE, "oracle.h")]
_LIB = os.path.join(_HERE, "liboracle.so")

_dp = C.POINTER(C.c_double)


def lib_path() -> str:
    return _LIB


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp (reading R15: no FMA contraction in the reference semantics)"""
    stale = (not os.path.exists(_LIB)) or any(os.path.getmtime(s) > os.path.getmtime(_LIB) for s in _SRC)
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall",
               _SRC[0], "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


class Oracle:
    """thin wrapper; one global context inside the library (like the five-call boundary)"""

    def __init__(self):
        build()
        L = C.CDLL(_LIB)
        L.oracle_init.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int]
        L.oracle_set_box.argtypes = [C.c_double] * 3
        L.oracle_set_state.argtypes = [_dp, _dp]
        L.oracle_get_state.argtypes = [_dp, _dp]
        L.oracle_step.argtypes = [C.c_int]
        L.oracle_step_fixed_dt.argtypes = [C.c_int, C.c_double]
        L.oracle_get_dt.restype = C.c_double
        L.oracle_get_time.restype = C.c_double
        L.oracle_set_threads.argtypes = [C.c_int]
        L.oracle_set_integrator.argtypes = [C.c_int]
        L.oracle_wenoz.argtypes = [_dp]
        L.oracle_wenoz.restype = C.c_double
        L.oracle_cons2prim.argtypes = [_dp, C.c_double, _dp]
        L.oracle_prim2cons.argtypes = [_dp, C.c_double, _dp]
        L.oracle_prim2cons.restype = None
        L.oracle_fast_speed.argtypes = [C.c_double] * 6
        L.oracle_fast_speed.restype = C.c_double
        L.oracle_plm_slope.argtypes = [C.c_double, C.c_double, C.c_int]
        L.oracle_plm_slope.restype = C.c_double
        L.oracle_physical_flux.argtypes = [_dp, C.c_double, C.c_double, _dp]
        L.oracle_physical_flux.restype = None
        L.oracle_hlld.argtypes = [_dp, _dp, C.c_double, C.c_double, _dp, _dp, _dp]
        L.oracle_debug_euler.argtypes = [C.c_double, _dp, _dp, _dp, _dp, _dp]
        L.oracle_set_divb.argtypes = [C.c_int]
        L.oracle_set_emf.argtypes = [C.c_int]
        L.oracle_hlld_uct.argtypes = [_dp, _dp, C.c_double, C.c_double, _dp, _dp, _dp, _dp]
        L.oracle_set_psi.argtypes = [_dp]
        L.oracle_get_psi.argtypes = [_dp]
        L.oracle_glm_interface.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.oracle_glm_interface.restype = None
        self.L = L
        self.shape = None

    # ---- the boundary calls
    def init(self, nx, ny, nz, ghost=2, gamma=5.0 / 3.0, cfl=0.4, limiter=0):
        rc = self.L.oracle_init(nx, ny, nz, ghost, gamma, cfl, limiter)
        if rc == 0:
            self.shape = (nx, ny, nz)
        return rc

    def set_box(self, Lx, Ly, Lz):
        return self.L.oracle_set_box(Lx, Ly, Lz)

    def nface(self):
        nx, ny, nz = self.shape
        return ((nx + 1) * ny * nz if nx > 1 else 0) + (nx * (ny + 1) * nz if ny > 1 else 0) \
            + (nx * ny * (nz + 1) if nz > 1 else 0)

    def set_state(self, U, Bface):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.size == 8 * np.prod(self.shape)
        if Bface is None:                        # GLM variant: no face fields
            return self.L.oracle_set_state(_ptr(U), None)
        Bface = np.ascontiguousarray(Bface, dtype=np.float64)
        assert Bface.size == self.nface()
        return self.L.oracle_set_state(_ptr(U), _ptr(Bface))

    def get_state(self, faces=True):
        nx, ny, nz = self.shape
        U = np.empty((8, nz, ny, nx))
        Bf = np.empty(self.nface()) if faces else None
        rc = self.L.oracle_get_state(_ptr(U), _ptr(Bf))
        assert rc == 0
        return U, Bf

    def step(self, n=1):
        return self.L.oracle_step(n)

    def step_fixed_dt(self, n, dt):
        return self.L.oracle_step_fixed_dt(n, dt)

    def get_dt(self):
        return self.L.oracle_get_dt()

    def get_time(self):
        return self.L.oracle_get_time()

    def set_threads(self, n):
        return self.L.oracle_set_threads(n)

    def get_threads(self):
        return self.L.oracle_get_threads()

    def set_integrator(self, order):
        return self.L.oracle_set_integrator(order)

    def finalize(self):
        return self.L.oracle_finalize()

    # ---- EMF average of the CT step: 0 = contact-mode upwinding with the continuous weight (R6), 1 = UCT-HLLD (R19)
    def set_emf(self, mode):
        return self.L.oracle_set_emf(mode)

    # ---- GLM divergence cleaning (R20)
    def set_divb(self, mode):
        return self.L.oracle_set_divb(mode)

    def set_psi(self, psi):
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        return self.L.oracle_set_psi(_ptr(psi))

    def get_psi(self):
        nx, ny, nz = self.shape
        psi = np.empty((nz, ny, nx))
        assert self.L.oracle_get_psi(_ptr(psi)) == 0
        return psi

    def glm_interface(self, BnL, BnR, psiL, psiR, ch):
        out = np.empty(2)
        self.L.oracle_glm_interface(BnL, BnR, psiL, psiR, ch, _ptr(out[0:1]), _ptr(out[1:2]))
        return float(out[0]), float(out[1])

    def load_glm(self, w, threads=None):
        """init + set_box + GLM mode + set_state (cell-centred B of w.U, psi = 0)"""
        if threads is not None:
            self.set_threads(threads)
        assert self.init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter) == 0
        assert self.set_box(*w.box) == 0
        assert self.set_divb(1) == 0
        assert self.set_state(w.U, None) == 0
        return self

    def load(self, w, threads=None):
        """init + set_box + set_state from a workloads.Workload"""
        if threads is not None:
            self.set_threads(threads)
        rc = self.init(w.nx, w.ny, w.nz, 2, w.gamma, w.cfl, w.limiter)
        assert rc == 0, rc
        assert self.set_box(*w.box) == 0
        assert self.set_state(w.U, w.Bface) == 0
        return self

    # ---- pieces
    def cons2prim(self, U, gamma):
        U = np.ascontiguousarray(U, dtype=np.float64)
        V = np.empty(8)
        rc = self.L.oracle_cons2prim(_ptr(U), gamma, _ptr(V))
        return rc, V

    def prim2cons(self, V, gamma):
        V = np.ascontiguousarray(V, dtype=np.float64)
        U = np.empty(8)
        self.L.oracle_prim2cons(_ptr(V), gamma, _ptr(U))
        return U

    def fast_speed(self, rho, p, Bn, Bt1, Bt2, gamma):
        return self.L.oracle_fast_speed(rho, p, Bn, Bt1, Bt2, gamma)

    def plm_slope(self, dm, dp, limiter):
        return self.L.oracle_plm_slope(dm, dp, limiter)

    def physical_flux(self, V7, Bn, gamma):
        V7 = np.ascontiguousarray(V7, dtype=np.float64)
        F = np.empty(8)
        self.L.oracle_physical_flux(_ptr(V7), Bn, gamma, _ptr(F))
        return F

    def hlld(self, VL, VR, Bn, gamma, debug=False):
        VL = np.ascontiguousarray(VL, dtype=np.float64)
        VR = np.ascontiguousarray(VR, dtype=np.float64)
        F = np.empty(8)
        w = C.c_double(0.0)
        dbg = np.zeros(72) if debug else None
        rc = self.L.oracle_hlld(_ptr(VL), _ptr(VR), Bn, gamma, _ptr(F), C.byref(w), _ptr(dbg))
        assert rc == 0
        return (F, w.value, dbg) if debug else (F, w.value)

    def hlld_uct(self, VL, VR, Bn, gamma):
        """flux, and uct = (a^L, d^L, d^R, vbar_t1, vbar_t2) of the UCT-HLLD average (R19)"""
        VL = np.ascontiguousarray(VL, dtype=np.float64)
        VR = np.ascontiguousarray(VR, dtype=np.float64)
        F = np.empty(8)
        uct = np.empty(5)
        w = C.c_double(0.0)
        dbg = np.zeros(72)
        rc = self.L.oracle_hlld_uct(_ptr(VL), _ptr(VR), Bn, gamma, _ptr(F), C.byref(w), _ptr(dbg), _ptr(uct))
        assert rc == 0
        return F, uct, dbg

    def debug_euler(self, dt, want=("U1", "Bf1", "F", "W", "E")):
        nx, ny, nz = self.shape
        N = nx * ny * nz
        out = {}
        if "U1" in want:
            out["U1"] = np.empty((8, nz, ny, nx))
        if "Bf1" in want:
            out["Bf1"] = np.empty(self.nface())
        if "F" in want:
            out["F"] = np.empty((3, 8, nz, ny, nx))
        if "W" in want:
            out["W"] = np.empty((3, nz, ny, nx))
        if "E" in want:
            out["E"] = np.empty((3, nz, ny, nx))
        rc = self.L.oracle_debug_euler(dt, _ptr(out.get("U1")), _ptr(out.get("Bf1")), _ptr(out.get("F")),
                                       _ptr(out.get("W")), _ptr(out.get("E")))
        out["rc"] = rc
        return out
