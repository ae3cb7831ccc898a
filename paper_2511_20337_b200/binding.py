"""Thin ctypes binding of libpluto_b200.so (include/pluto.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device
memory (the workspace the library computes in) and the stream it launches on.  There is no CPU
fallback: a missing library or a missing device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(_HERE, "libpluto_b200.so")

OK, EINVAL, ESTATE, ECUDA, EPHYS, ENOMEM = 0, -1, -2, -3, -4, -5
MINMOD, MC, WENOZ = 0, 1, 2
OPT_GRAPH = 1
OPT_FUSE_XY = 2
OPT_CT_TMA = 3
OPT_RK_ORDER = 4
OPT_DIVB = 5
DIVB_CT, DIVB_GLM = 0, 1
OPT_EMF = 6
EMF_CONTACT, EMF_UCT_HLLD = 0, 1

# every symbol include/pluto.h and include/pluto_debug.h declare
SYMBOLS = [
    "pluto_init", "pluto_set_state", "pluto_step", "pluto_get_dt", "pluto_get_state",
    "pluto_set_box", "pluto_step_fixed_dt", "pluto_get_time", "pluto_set_stream",
    "pluto_workspace_bytes", "pluto_set_workspace", "pluto_finalize", "pluto_last_error",
    "pluto_device_count", "pluto_step_async", "pluto_sync", "pluto_launch_count",
    "pluto_set_option", "pluto_debug_euler", "pluto_profile", "pluto_profile_get", "pluto_kernel_name",
    "pluto_probe_fp64_gflops",
    "pluto_init_slabs", "pluto_workspace_bytes_slabs", "pluto_local_planes", "pluto_export_slab",
    "pluto_attach_peer", "pluto_fill_ghosts", "pluto_slab_planes", "pluto_set_psi", "pluto_get_psi", "pluto_step_begin", "pluto_dt_max_bits", "pluto_step_stage",
    "pluto_cfl_dt_noalloc", "pluto_graph_captures",
]
NOALLOC_MAX_ROWS = 131072          # PLUTO_NOALLOC_MAX_ROWS of include/pluto.h


class PlutoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"pluto error {code}: {msg}")
        self.code = code


def load_library(build_if_missing: bool = True) -> C.CDLL:
    if build_if_missing:
        from . import build as _build
        _build.build()
    if not os.path.exists(LIB):
        raise RuntimeError(f"{LIB} is missing: build it with `python -m paper_2511_20337_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB)
    vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
    L.pluto_init.argtypes = [i32, i32, i32, i32, dbl, dbl, i32]
    L.pluto_set_state.argtypes = [vp, vp]
    L.pluto_step.argtypes = [i32]
    L.pluto_get_dt.restype = dbl
    L.pluto_get_state.argtypes = [vp, vp]
    L.pluto_set_box.argtypes = [dbl, dbl, dbl]
    L.pluto_step_fixed_dt.argtypes = [i32, dbl]
    L.pluto_get_time.restype = dbl
    L.pluto_set_stream.argtypes = [vp]
    L.pluto_workspace_bytes.argtypes = [i32, i32, i32, i32]
    L.pluto_workspace_bytes.restype = C.c_size_t
    L.pluto_set_workspace.argtypes = [vp, C.c_size_t]
    L.pluto_last_error.restype = C.c_char_p
    L.pluto_step_async.argtypes = [i32]
    L.pluto_launch_count.restype = C.c_longlong
    L.pluto_graph_captures.restype = C.c_longlong
    L.pluto_set_option.argtypes = [i32, i32]
    L.pluto_debug_euler.argtypes = [dbl, vp, vp, vp, vp, vp]
    L.pluto_profile.argtypes = [i32]
    L.pluto_profile_get.argtypes = [i32, C.POINTER(dbl), C.POINTER(C.c_longlong)]
    L.pluto_kernel_name.argtypes = [i32]
    L.pluto_kernel_name.restype = C.c_char_p
    L.pluto_probe_fp64_gflops.restype = dbl
    L.pluto_init_slabs.argtypes = [i32, i32, i32, i32, i32, i32, i32, dbl, dbl, i32]
    L.pluto_workspace_bytes_slabs.argtypes = [i32] * 8
    L.pluto_workspace_bytes_slabs.restype = C.c_size_t
    L.pluto_local_planes.argtypes = [C.POINTER(i32), C.POINTER(i32)]
    L.pluto_slab_planes.argtypes = [i32, i32, i32, C.POINTER(i32), C.POINTER(i32)]
    L.pluto_export_slab.argtypes = [i32, vp, C.POINTER(vp), C.POINTER(C.c_longlong), C.POINTER(i32)]
    L.pluto_attach_peer.argtypes = [i32, vp, vp, C.c_longlong, i32]
    L.pluto_step_begin.argtypes = [dbl]
    L.pluto_dt_max_bits.restype = vp
    L.pluto_step_stage.argtypes = [i32, i32]
    L.pluto_set_psi.argtypes = [vp]
    L.pluto_get_psi.argtypes = [vp]
    L.pluto_cfl_dt_noalloc.argtypes = [vp, i32, i32, i32, dbl, dbl, dbl, dbl, dbl, vp, vp]
    return L


def _addr(a):
    """host numpy array or CUDA torch tensor -> raw address (the library tells host from device)"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float64 and a.flags.c_contiguous
        return a.ctypes.data
    assert a.dtype.is_floating_point and a.element_size() == 8 and a.is_contiguous()
    return a.data_ptr()


class Pluto:
    """pluto_* calls with the same names; arrays are numpy (host) or torch CUDA tensors (device)"""

    def __init__(self, device: int = 0):
        import torch
        self.L = load_library()
        if self.L.pluto_device_count() < 1 or not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2511_20337_b200 has no CPU fallback")
        self.torch = torch
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.Stream(device=self.device)
        self._check(self.L.pluto_set_stream(self.stream.cuda_stream))
        self.workspace = None
        self.shape = None
        self.rk_order = 2

    def _check(self, rc):
        if rc != 0:
            raise PlutoError(rc, self.L.pluto_last_error().decode())
        return rc

    # ---- the five calls
    def init(self, nx, ny, nz, ghost=2, gamma=5.0 / 3.0, cfl=0.4, limiter=MINMOD, nslab=1):
        """nslab > 1: the box cut into nslab z slabs, all of them on this GPU (pluto_init_slabs)"""
        need = self.L.pluto_workspace_bytes_slabs(nslab, 0, nslab, nx, ny, nz, ghost, self.rk_order)
        if need == 0:
            raise PlutoError(EINVAL, "bad grid")
        self.L.pluto_finalize()
        if self.workspace is None or self.workspace.numel() < need:
            self.workspace = None
            self.workspace = self.torch.empty(need, dtype=self.torch.uint8, device=self.device)
        self.torch.cuda.current_stream().synchronize()
        self._check(self.L.pluto_set_workspace(self.workspace.data_ptr(), self.workspace.numel()))
        if nslab == 1:
            self._check(self.L.pluto_init(nx, ny, nz, ghost, gamma, cfl, limiter))
        else:
            self._check(self.L.pluto_init_slabs(nslab, 0, nslab, nx, ny, nz, ghost, gamma, cfl, limiter))
        self.shape = (nx, ny, nz)
        return 0

    def nface(self):
        nx, ny, nz = self.shape
        return (nx + 1) * ny * nz + nx * (ny + 1) * nz + (nx * ny * (nz + 1) if nz > 1 else 0)

    def set_state(self, U, Bface):
        if isinstance(U, np.ndarray):
            U = np.ascontiguousarray(U, dtype=np.float64)
            Bface = np.ascontiguousarray(Bface, dtype=np.float64)
        else:
            self.torch.cuda.current_stream().synchronize()
        assert U.size == 8 * int(np.prod(self.shape)) if isinstance(U, np.ndarray) else U.numel() == 8 * int(np.prod(self.shape))
        return self._check(self.L.pluto_set_state(_addr(U), _addr(Bface)))

    def step(self, nsteps=1):
        return self._check(self.L.pluto_step(nsteps))

    def get_dt(self):
        return self.L.pluto_get_dt()

    def get_state(self, out_U=None, out_B=None, device=False):
        nx, ny, nz = self.shape
        if out_U is None:
            if device:
                out_U = self.torch.empty((8, nz, ny, nx), dtype=self.torch.float64, device=self.device)
                out_B = self.torch.empty(self.nface(), dtype=self.torch.float64, device=self.device)
                self.torch.cuda.current_stream().synchronize()
            else:
                out_U = np.empty((8, nz, ny, nx))
                out_B = np.empty(self.nface())
        self._check(self.L.pluto_get_state(_addr(out_U), _addr(out_B)))
        return out_U, out_B

    # ---- extensions
    def set_box(self, Lx, Ly, Lz):
        return self._check(self.L.pluto_set_box(Lx, Ly, Lz))

    def step_fixed_dt(self, nsteps, dt):
        return self._check(self.L.pluto_step_fixed_dt(nsteps, dt))

    def get_time(self):
        return self.L.pluto_get_time()

    def step_async(self, nsteps):
        return self._check(self.L.pluto_step_async(nsteps))

    def sync(self):
        return self._check(self.L.pluto_sync())

    def launch_count(self):
        return self.L.pluto_launch_count()

    def graph_captures(self):
        return self.L.pluto_graph_captures()

    def set_option(self, opt, value):
        return self.L.pluto_set_option(opt, value)

    def set_integrator(self, order):
        """2: SSP-RK2 (default), 3: SSP-RK3 of Eq. 5; returns the previous order"""
        old = self.L.pluto_set_option(OPT_RK_ORDER, order)
        if old < 0:
            raise PlutoError(old, self.L.pluto_last_error().decode())
        self.rk_order = order
        return old

    def profile(self, on):
        return self._check(self.L.pluto_profile(1 if on else 0))

    def profile_report(self):
        """{kernel name: (total ms, launches)} accumulated since profile(True)"""
        out, k = {}, 0
        while True:
            name = self.L.pluto_kernel_name(k)
            if name is None:
                return out
            ms, cnt = C.c_double(0.0), C.c_longlong(0)
            self._check(self.L.pluto_profile_get(k, C.byref(ms), C.byref(cnt)))
            out[name.decode()] = (ms.value, cnt.value)
            k += 1

    def probe_fp64_gflops(self):
        return self.L.pluto_probe_fp64_gflops()

    def finalize(self):
        return self.L.pluto_finalize()

    def cfl_dt_noalloc(self, U, box, gamma, cfl, out, stream=None):
        """pluto_cfl_dt_noalloc: the CFL dt of a state the caller holds, for callers whose memory is all in their
        own pool (the library allocates nothing here; its scratch is a fixed array inside the library, which is why
        ny * nz may not exceed NOALLOC_MAX_ROWS).  U: CUDA float64 tensor [8][nz][ny][nx] as get_state returns it;
        out: CUDA float64 tensor of 3 (dt, max signal speed / dx, unphysical flag), written asynchronously on
        `stream` (a torch.cuda.Stream; default: this object's stream) -- synchronise it before reading out.
        Calls that could overlap on the GPU share the scratch and must be ordered by the caller."""
        assert U.is_cuda and out.is_cuda and U.dim() == 4 and U.shape[0] == 8 and out.numel() >= 3
        _, nz, ny, nx = U.shape
        s = self.stream if stream is None else stream
        return self._check(self.L.pluto_cfl_dt_noalloc(_addr(U), nx, ny, nz, box[0], box[1], box[2], gamma, cfl,
                                                       _addr(out), s.cuda_stream))

    def set_emf(self, mode):
        """EMF average of the CT step: EMF_CONTACT (default, reading R6) or EMF_UCT_HLLD (reading R19)"""
        old = self.L.pluto_set_option(OPT_EMF, mode)
        if old < 0:
            raise ValueError(self.last_error())
        return old

    # ---- GLM divergence cleaning (PLUTO_OPT_DIVB; reading R20)
    def set_divb(self, mode):
        """divergence control of the NEXT init: DIVB_CT (default) or DIVB_GLM"""
        old = self.L.pluto_set_option(OPT_DIVB, mode)
        if old < 0:
            raise PlutoError(old, self.L.pluto_last_error().decode())
        return old

    def load_glm(self, w, ghost=2):
        """init (GLM variant) + set_box + set_state from a workloads.Workload: cell-centred B of w.U, psi = 0"""
        self.set_divb(DIVB_GLM)
        try:
            self.init(w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter)
        finally:
            self.set_divb(DIVB_CT)
        self.set_box(*w.box)
        U = np.ascontiguousarray(w.U, dtype=np.float64)
        return self._check(self.L.pluto_set_state(_addr(U), None))

    def get_state_glm(self):
        nx, ny, nz = self.shape
        U = np.empty((8, nz, ny, nx))
        self._check(self.L.pluto_get_state(_addr(U), None))
        return U

    def set_psi(self, psi):
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        return self._check(self.L.pluto_set_psi(_addr(psi)))

    def get_psi(self):
        nx, ny, nz = self.shape
        psi = np.empty((nz, ny, nx))
        self._check(self.L.pluto_get_psi(_addr(psi)))
        return psi

    def load(self, w, ghost=None, nslab=1):
        """init + set_box + set_state from a workloads.Workload (host arrays)"""
        if ghost is None:
            ghost = 3 if w.limiter == WENOZ else 2
        self.init(w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter, nslab=nslab)
        self.set_box(*w.box)
        self.set_state(w.U, w.Bface)
        return self

    def debug_euler(self, dt, want=("U1", "Bf1", "W", "Fem", "E")):
        nx, ny, nz = self.shape
        out = {}
        if "U1" in want:
            out["U1"] = np.empty((8, nz, ny, nx))
        if "Bf1" in want:
            out["Bf1"] = np.empty(self.nface())
        if "W" in want:
            out["W"] = np.empty((3, nz, ny, nx))
        if "Fem" in want:
            out["Fem"] = np.empty((3, 2, nz, ny, nx))
        if "E" in want:
            out["E"] = np.empty((3, nz, ny, nx))
        rc = self.L.pluto_debug_euler(dt, _addr(out.get("U1")), _addr(out.get("Bf1")), _addr(out.get("W")),
                                      _addr(out.get("Fem")), _addr(out.get("E")))
        out["rc"] = rc
        return out
