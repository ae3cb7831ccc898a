"""One z slab of the periodic box per process, one process per GPU: the domain-decomposed step of
section 3.4 "Multi GPU communication" (Fig. 4) on an NVLink / NVSwitch node.

What crosses GPUs, per Runge-Kutta stage, is the `ghost` planes of the 8 state arrays on each side of a
slab.  The paper packs them into buffers and posts MPI_Isend / MPI_Irecv pairs (Fig. 4);
here the ghost-fill KERNEL of a slab reads the planes straight out of its neighbours' device memory
(CUDA IPC mapping, peer loads over NVLink): no pack / unpack kernels, no staging copies, and the same
kernel whether the neighbour slab lives in this process or on another GPU.  The only collectives are one
MAX all-reduce of 8 bytes per step (the CFL dt, a8) and one barrier per stage (a slab's ghost fill may
start when its neighbours have finished the previous stage); both are issued on the library's stream, so
the host never waits.

`torch.distributed` is plumbing: it carries the IPC handles once and issues those two collectives.  All
arithmetic stays in the kernels behind the C ABI (pluto_init_slabs ... pluto_step_stage, include/pluto.h).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import binding as B


def neighbour_ranks(rank: int, world: int):
    """ranks holding the slab below and the slab above (periodic in z)"""
    return (rank - 1) % world, (rank + 1) % world


def slab_planes(nz: int, nslab: int, slab: int):
    """(first plane, planes) of slab `slab`: the library's own partition (pluto_slab_planes; no device needed)"""
    L = B.load_library()
    k0, n = C.c_int(0), C.c_int(0)
    rc = L.pluto_slab_planes(nz, nslab, slab, k0, n)
    if rc != 0:
        raise B.PlutoError(rc, L.pluto_last_error().decode())
    return k0.value, n.value


def local_part(U, Bface, nx, ny, nz, k0, nzl):
    """the planes [k0, k0 + nzl) of a whole-box state in the layouts of pluto_set_state: U[8][nzl][ny][nx] and
    [bx: nzl*ny*(nx+1)] [by: nzl*(ny+1)*nx] [bz: (nzl+1)*ny*nx] (the last bz plane is the upper boundary face)"""
    from . import workloads as wl
    f = wl.split_faces(Bface, nx, ny, nz)
    Ul = np.ascontiguousarray(np.asarray(U).reshape(8, nz, ny, nx)[:, k0:k0 + nzl])
    parts = [f["bx"][k0:k0 + nzl].ravel(), f["by"][k0:k0 + nzl].ravel(), f["bz"][k0:k0 + nzl + 1].ravel()]
    return Ul, np.ascontiguousarray(np.concatenate(parts))


def join_parts(parts, nx, ny, nz):
    """inverse of local_part over all slabs: [(k0, nzl, U_local, B_local), ...] -> whole-box (U, Bface)"""
    from . import workloads as wl
    U = np.empty((8, nz, ny, nx))
    bx, by, bz = np.empty((nz, ny, nx + 1)), np.empty((nz, ny + 1, nx)), np.empty((nz + 1, ny, nx))
    for k0, nzl, Ul, Bl in parts:
        U[:, k0:k0 + nzl] = Ul.reshape(8, nzl, ny, nx)
        n1, n2 = nzl * ny * (nx + 1), nzl * (ny + 1) * nx
        bx[k0:k0 + nzl] = Bl[:n1].reshape(nzl, ny, nx + 1)
        by[k0:k0 + nzl] = Bl[n1:n1 + n2].reshape(nzl, ny + 1, nx)
        bz[k0:k0 + nzl + 1] = Bl[n1 + n2:].reshape(nzl + 1, ny, nx)
    return U, wl.join_faces({"bx": bx, "by": by, "bz": bz}, nx, ny, nz)


class _DevicePtr:
    """a raw device address as a CUDA array (for torch.as_tensor)"""

    def __init__(self, ptr, count, typestr):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 3, "strides": None}


class SlabPluto:
    """pluto_* calls on the slab of this rank.  `dist` is an initialised torch.distributed module (backend
    nccl: collectives run on the device, ordered with the library's stream; backend gloo: the host waits
    for the stream around each collective -- used by the tests, where two processes share one GPU)."""

    def __init__(self, dist, device: int = 0):
        import torch
        self.torch, self.dist = torch, dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()
        self.L = B.load_library()
        if self.L.pluto_device_count() < 1 or not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_2511_20337_b200 has no CPU fallback")
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.Stream(device=self.device)
        self._check(self.L.pluto_set_stream(self.stream.cuda_stream))
        self.on_device = dist.get_backend() == "nccl"
        self.rk_order = 2
        self.shape = None
        self._token = torch.zeros(1, dtype=torch.int32, device=self.device) if self.on_device else None

    def _check(self, rc):
        if rc != 0:
            raise B.PlutoError(rc, self.L.pluto_last_error().decode())
        return rc

    # ---- collectives (plumbing)
    def barrier(self):
        """every rank's enqueued work is complete before anything enqueued after this call starts"""
        if self.on_device:
            with self.torch.cuda.stream(self.stream):
                self.dist.all_reduce(self._token)
        else:
            self.stream.synchronize()
            self.dist.barrier()

    def _allreduce_max_bits(self):
        """MAX over the ranks of the 8 bytes at pluto_dt_max_bits(): bit patterns of positive doubles order
        like signed 64-bit integers"""
        t = self.torch.as_tensor(_DevicePtr(self.L.pluto_dt_max_bits(), 1, "<i8"), device=self.device)
        if self.on_device:
            with self.torch.cuda.stream(self.stream):
                self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        else:
            self.stream.synchronize()
            h = t.cpu()
            self.dist.all_reduce(h, op=self.dist.ReduceOp.MAX)
            with self.torch.cuda.stream(self.stream):
                t.copy_(h.to(self.device))
            self.stream.synchronize()

    # ---- set-up
    def set_integrator(self, order):
        old = self.L.pluto_set_option(B.OPT_RK_ORDER, order)
        if old < 0:
            raise B.PlutoError(old, self.L.pluto_last_error().decode())
        self.rk_order = order
        return old

    def init(self, nx, ny, nz, ghost=2, gamma=5.0 / 3.0, cfl=0.4, limiter=B.MINMOD, box=None):
        """nz = planes of the WHOLE box; this rank holds slab `rank` of `world`"""
        self.barrier()                                   # nobody still reads the memory about to be freed
        self.L.pluto_finalize()
        self._check(self.L.pluto_set_workspace(None, 0))          # the library allocates: IPC needs cudaMalloc'ed memory
        self._check(self.L.pluto_init_slabs(self.world, self.rank, 1, nx, ny, nz, ghost, gamma, cfl, limiter))
        if box is not None:
            self._check(self.L.pluto_set_box(*box))
        k0, nzl = C.c_int(0), C.c_int(0)
        self._check(self.L.pluto_local_planes(k0, nzl))
        self.k0, self.nzl, self.shape = k0.value, nzl.value, (nx, ny, nz)
        # exchange the slabs' IPC handles and attach the two neighbours
        handle = (C.c_ubyte * 64)()
        sa, planes = C.c_longlong(0), C.c_int(0)
        self._check(self.L.pluto_export_slab(0, handle, None, sa, planes))
        mine = (bytes(handle), sa.value, planes.value)
        everyone = [None] * self.world
        self.dist.all_gather_object(everyone, mine)
        self.peers = everyone
        for side, peer in enumerate(neighbour_ranks(self.rank, self.world)):
            if self.world == 1:
                break                                    # one slab: the library wired it to itself
            h, psa, pn = everyone[peer]
            buf = (C.c_ubyte * 64).from_buffer_copy(h)
            self._check(self.L.pluto_attach_peer(side, buf, None, psa, pn))
        self.barrier()
        return 0

    def nface_local(self):
        nx, ny, _ = self.shape
        return self.nzl * ny * (nx + 1) + self.nzl * (ny + 1) * nx + (self.nzl + 1) * ny * nx

    def set_state(self, U_local, B_local):
        """the planes this rank holds, layouts of local_part()"""
        U_local = np.ascontiguousarray(U_local, dtype=np.float64)
        B_local = np.ascontiguousarray(B_local, dtype=np.float64)
        assert U_local.size == 8 * self.nzl * self.shape[0] * self.shape[1] and B_local.size == self.nface_local()
        self._check(self.L.pluto_set_state(B._addr(U_local), B._addr(B_local)))
        self.barrier()                                   # every rank's interior is in place
        self._check(self.L.pluto_fill_ghosts())
        self.barrier()
        return 0

    def load(self, w, ghost=None):
        """init + set_state of this rank's planes of a whole-box workloads.Workload"""
        if ghost is None:
            ghost = 3 if w.limiter == B.WENOZ else 2
        self.init(w.nx, w.ny, w.nz, ghost, w.gamma, w.cfl, w.limiter, box=w.box)
        Ul, Bl = local_part(w.U, w.Bface, w.nx, w.ny, w.nz, self.k0, self.nzl)
        return self.set_state(Ul, Bl)

    # ---- the step in phases (include/pluto.h)
    def step_async(self, nsteps=1, fixed_dt=None):
        fixed = fixed_dt is not None
        for _ in range(nsteps):
            self._check(self.L.pluto_step_begin(float(fixed_dt) if fixed else 0.0))
            if fixed:
                self.barrier()                           # the neighbours have finished the previous step
            else:
                self._allreduce_max_bits()               # ... which the dt all-reduce implies as well
            for s in range(self.rk_order):
                if s > 0:
                    self.barrier()                       # the neighbours have finished stage s - 1
                self._check(self.L.pluto_step_stage(s, 1 if fixed else 0))

    def sync(self):
        return self._check(self.L.pluto_sync())

    def step(self, nsteps=1, fixed_dt=None):
        self.step_async(nsteps, fixed_dt)
        return self.sync()

    def get_dt(self):
        return self.L.pluto_get_dt()

    def get_time(self):
        return self.L.pluto_get_time()

    def launch_count(self):
        return self.L.pluto_launch_count()

    def get_state(self):
        """(U_local, B_local) of this rank's planes; the upper boundary b_z face comes from the slab above"""
        self.barrier()
        nx, ny, _ = self.shape
        U = np.empty((8, self.nzl, ny, nx))
        Bf = np.empty(self.nface_local())
        self._check(self.L.pluto_get_state(B._addr(U), B._addr(Bf)))
        return U, Bf

    def finalize(self):
        self.barrier()
        return self.L.pluto_finalize()
