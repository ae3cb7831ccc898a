"""Seeded synthetic initial conditions (the five BASELINE.json configs + small test problems).

This module serves BOTH the CUDA path and the oracle and therefore holds none of the method's
arithmetic: it only writes initial data -- analytic fields sampled on the mesh, the definition of
the conserved variables (Eq. 2-3), a discrete curl of a vector potential so that
the face field is divergence-free, and a counter-based noise generator.  It imports neither the
binding nor anything under oracle/.

The configs stand in for the paper's own analytic workloads: the Orszag-Tang vortex
(here in its classic 2D form) and the circularly polarised Alfven wave
(Eq. 10 with the e_z typo fixed, reading R2), plus a 3D MHD blast.

Layouts are those of include/pluto.h: U[8][nz][ny][nx]; Bface = bx[nz][ny][nx+1] ++ by[nz][ny+1][nx]
(++ bz[nz+1][ny][nx] in 3D).
"""
from __future__ import annotations

import dataclasses
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def counter_noise(seed: int, n: int, start: int = 0) -> np.ndarray:
    """u[c] in [0,1) for linear cell index c = start..start+n-1: a 64-bit integer mixer keyed by (seed, c).

    Stateless (counter based), so any sub-range can be regenerated independently."""
    with np.errstate(over="ignore"):
        z = np.arange(start, start + n, dtype=np.uint64) + np.uint64(seed) * np.uint64(0x9E3779B97F4A7C15)
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


@dataclasses.dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    box: tuple            # (Lx, Ly, Lz)
    gamma: float
    cfl: float
    limiter: int          # 0 minmod, 1 MC
    nsteps: int           # steps of the paper-shaped run (t_end for the wave: see t_end)
    U: np.ndarray         # (8, nz, ny, nx) float64
    Bface: np.ndarray     # flat float64
    t_end: float | None = None
    seed: int = 0

    @property
    def zones(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def ndim(self) -> int:
        return 3 if self.nz > 1 else (2 if self.ny > 1 else 1)


def face_shapes(nx, ny, nz):
    """shapes of the face arrays present for this grid (a family exists iff its n_d > 1)"""
    out = []
    if nx > 1:
        out.append(("bx", (nz, ny, nx + 1)))
    if ny > 1:
        out.append(("by", (nz, ny + 1, nx)))
    if nz > 1:
        out.append(("bz", (nz + 1, ny, nx)))
    return out


def split_faces(Bface, nx, ny, nz):
    """flat Bface -> dict of views {'bx': (nz,ny,nx+1), ...}"""
    out, off = {}, 0
    for name, shp in face_shapes(nx, ny, nz):
        n = int(np.prod(shp))
        out[name] = Bface[off:off + n].reshape(shp)
        off += n
    assert off == Bface.size
    return out


def join_faces(faces, nx, ny, nz):
    return np.concatenate([np.ascontiguousarray(faces[name], dtype=np.float64).ravel()
                           for name, _ in face_shapes(nx, ny, nz)]) if face_shapes(nx, ny, nz) else np.zeros(0)


def cell_centres(n, L):
    return (np.arange(n) + 0.5) * (L / n)


def face_positions(n, L):
    return np.arange(n + 1) * (L / n)


def conserved_from_fields(rho, v, Bcell, p, gamma):
    """U of Eq. 2-3 from point values; every argument broadcast to (nz,ny,nx)"""
    shp = rho.shape
    U = np.empty((8,) + shp, dtype=np.float64)
    U[0] = rho
    for d in range(3):
        U[1 + d] = rho * v[d]
        U[4 + d] = Bcell[d]
    U[7] = p / (gamma - 1.0) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2) \
        + 0.5 * (Bcell[0] ** 2 + Bcell[1] ** 2 + Bcell[2] ** 2)
    return U


def cell_mean_of_faces(faces, nx, ny, nz, Bcell):
    """cell-centred B of each active direction = mean of its two faces"""
    if "bx" in faces:
        Bcell[0] = 0.5 * (faces["bx"][:, :, :-1] + faces["bx"][:, :, 1:])
    if "by" in faces:
        Bcell[1] = 0.5 * (faces["by"][:, :-1, :] + faces["by"][:, 1:, :])
    if "bz" in faces:
        Bcell[2] = 0.5 * (faces["bz"][:-1, :, :] + faces["bz"][1:, :, :])
    return Bcell


# --------------------------------------------------------------------------- Orszag-Tang (C0, C2)

def orszag_tang_2d(n=128, nsteps=100, seed=20337, noise=1e-3, gamma=5.0 / 3.0, cfl=0.4, limiter=0,
                   name=None, ny=None):
    nx = n
    ny = n if ny is None else ny
    nz = 1
    Lx, Ly = 1.0, ny / nx
    dx, dy = Lx / nx, Ly / ny
    x, y = cell_centres(nx, Lx), cell_centres(ny, Ly)
    xf, yf = face_positions(nx, Lx), face_positions(ny, Ly)
    B0 = 1.0 / np.sqrt(4.0 * np.pi)
    two_pi = 2.0 * np.pi

    def Az(xx, yy):
        return B0 * (np.cos(two_pi * yy) / two_pi + np.cos(2.0 * two_pi * xx) / (2.0 * two_pi))

    A = Az(xf[None, :], yf[:, None])                   # corners (ny+1, nx+1)
    bx = (A[1:, :] - A[:-1, :]) / dy                   # (ny, nx+1):  dAz/dy
    by = -(A[:, 1:] - A[:, :-1]) / dx                  # (ny+1, nx): -dAz/dx
    faces = {"bx": bx[None], "by": by[None]}
    rho0 = 25.0 / (36.0 * np.pi)
    p0 = 5.0 / (12.0 * np.pi)
    u = counter_noise(seed, nx * ny * nz).reshape(nz, ny, nx)
    rho = rho0 * (1.0 + noise * (2.0 * u - 1.0))
    X = np.broadcast_to(x[None, None, :], (nz, ny, nx))
    Y = np.broadcast_to(y[None, :, None], (nz, ny, nx))
    v = [-np.sin(two_pi * Y), np.sin(two_pi * X), np.zeros((nz, ny, nx))]
    Bc = cell_mean_of_faces(faces, nx, ny, nz, [None, None, np.zeros((nz, ny, nx))])
    U = conserved_from_fields(rho, v, Bc, np.full((nz, ny, nx), p0), gamma)
    return Workload(name or f"orszag_tang_2d_{nx}x{ny}", nx, ny, nz, (Lx, Ly, Ly), gamma, cfl, limiter,
                    nsteps, U, join_faces(faces, nx, ny, nz), seed=seed)


# --------------------------------------------------------------------------- 3D Orszag-Tang vortex (the paper's own benchmark)

def orszag_tang_3d(n=64, seed=4155, noise=0.0, gamma=5.0 / 3.0, cfl=0.3, limiter=1, name=None, shape=None):
    """The 3D Orszag-Tang vortex of PAPER.md:254-258 (section 4.1): unit periodic cube, rho = 25/9, p = 5/3,
    v = (-zeta sin 2 pi y, zeta sin 2 pi x, 0.2 sin 2 pi z), zeta = 1 + sin(2 pi z)/5, B = (-sin 2 pi y, sin 4 pi x, 0).
    Face B is the discrete curl of A_z = cos(2 pi y)/(2 pi) + cos(4 pi x)/(4 pi); optional seeded density noise."""
    nx, ny, nz = (n, n, n) if shape is None else shape
    L = (1.0, ny / nx, nz / nx)
    dx, dy = L[0] / nx, L[1] / ny
    x, y, z = cell_centres(nx, L[0]), cell_centres(ny, L[1]), cell_centres(nz, L[2])
    xf, yf = face_positions(nx, L[0]), face_positions(ny, L[1])
    two_pi = 2.0 * np.pi
    A = np.cos(two_pi * yf[:, None]) / two_pi + np.cos(2.0 * two_pi * xf[None, :]) / (2.0 * two_pi)   # (ny+1, nx+1)
    bx = (A[1:, :] - A[:-1, :]) / dy
    by = -(A[:, 1:] - A[:, :-1]) / dx
    faces = {"bx": np.broadcast_to(bx[None], (nz, ny, nx + 1)).copy(),
             "by": np.broadcast_to(by[None], (nz, ny + 1, nx)).copy(),
             "bz": np.zeros((nz + 1, ny, nx))}
    shp = (nz, ny, nx)
    X = np.broadcast_to(x[None, None, :], shp)
    Y = np.broadcast_to(y[None, :, None], shp)
    Z = np.broadcast_to(z[:, None, None], shp)
    zeta = 1.0 + np.sin(two_pi * Z) / 5.0
    v = [-zeta * np.sin(two_pi * Y), zeta * np.sin(two_pi * X), 0.2 * np.sin(two_pi * Z)]
    rho = np.full(shp, 25.0 / 9.0)
    if noise:
        rho = rho * (1.0 + noise * (2.0 * counter_noise(seed, nx * ny * nz).reshape(shp) - 1.0))
    Bc = cell_mean_of_faces(faces, nx, ny, nz, [None, None, None])
    U = conserved_from_fields(rho, v, Bc, np.full(shp, 5.0 / 3.0), gamma)
    return Workload(name or f"orszag_tang_3d_{nx}x{ny}x{nz}", nx, ny, nz, L, gamma, cfl, limiter, 0, U,
                    join_faces(faces, nx, ny, nz), t_end=0.5, seed=seed)


# --------------------------------------------------------------------------- CP Alfven wave (C1)

def cp_alfven_3d(nx=64, seed=2511, noise=1e-6, gamma=5.0 / 3.0, cfl=0.4, limiter=1, amp=0.1, name=None):
    """Oblique circularly polarised Alfven wave, box 3 x 1.5 x 1.5, grid nx x nx/2 x nx/2.

    Wave frame e1 = (1,2,2)/3 = k/|k| for k = 2 pi (1/Lx, 1/Ly, 1/Lz); wavelength 1;
    Eq. 10 with the second velocity term along e3 (R2)."""
    ny = nz = nx // 2
    Lx, Ly, Lz = 3.0, 1.5, 1.5
    d = (Lx / nx, Ly / ny, Lz / nz)
    e1 = np.array([1.0, 2.0, 2.0]) / 3.0
    e2 = np.array([-2.0, 1.0, 0.0]) / np.sqrt(5.0)
    e3 = np.array([-2.0, -4.0, 5.0]) / (3.0 * np.sqrt(5.0))
    two_pi = 2.0 * np.pi

    def phase(xx, yy, zz):
        return two_pi * (e1[0] * xx + e1[1] * yy + e1[2] * zz)

    xc, yc, zc = cell_centres(nx, Lx), cell_centres(ny, Ly), cell_centres(nz, Lz)
    xf, yf, zf = face_positions(nx, Lx), face_positions(ny, Ly), face_positions(nz, Lz)

    def Avec(comp, xx, yy, zz):
        ph = phase(xx, yy, zz)
        return (amp / two_pi) * (np.sin(ph) * e2[comp] + np.cos(ph) * e3[comp])

    # vector potential at edge midpoints: A_x at (x_c, y_f, z_f), A_y at (x_f, y_c, z_f), A_z at (x_f, y_f, z_c)
    Ax = Avec(0, xc[None, None, :], yf[None, :, None], zf[:, None, None])    # (nz+1, ny+1, nx)
    Ay = Avec(1, xf[None, None, :], yc[None, :, None], zf[:, None, None])    # (nz+1, ny, nx+1)
    Az = Avec(2, xf[None, None, :], yf[None, :, None], zc[:, None, None])    # (nz, ny+1, nx+1)
    bx = (Az[:, 1:, :] - Az[:, :-1, :]) / d[1] - (Ay[1:, :, :] - Ay[:-1, :, :]) / d[2]    # (nz, ny, nx+1)
    by = (Ax[1:, :, :] - Ax[:-1, :, :]) / d[2] - (Az[:, :, 1:] - Az[:, :, :-1]) / d[0]    # (nz, ny+1, nx)
    bz = (Ay[:, :, 1:] - Ay[:, :, :-1]) / d[0] - (Ax[:, 1:, :] - Ax[:, :-1, :]) / d[1]    # (nz+1, ny, nx)
    faces = {"bx": bx + e1[0], "by": by + e1[1], "bz": bz + e1[2]}          # B_parallel = 1 along e1
    shp = (nz, ny, nx)
    X = np.broadcast_to(xc[None, None, :], shp)
    Y = np.broadcast_to(yc[None, :, None], shp)
    Z = np.broadcast_to(zc[:, None, None], shp)
    ph = phase(X, Y, Z)
    v = [amp * (np.sin(ph) * e2[c] + np.cos(ph) * e3[c]) for c in range(3)]
    u = counter_noise(seed, nx * ny * nz).reshape(shp)
    p = 0.1 * (1.0 + noise * (2.0 * u - 1.0))
    Bc = cell_mean_of_faces(faces, nx, ny, nz, [None, None, None])
    U = conserved_from_fields(np.ones(shp), v, Bc, p, gamma)
    return Workload(name or f"cp_alfven_3d_{nx}x{ny}x{nz}", nx, ny, nz, (Lx, Ly, Lz), gamma, cfl, limiter,
                    0, U, join_faces(faces, nx, ny, nz), t_end=1.0, seed=seed)


def cp_alfven_1d(nx=64, gamma=5.0 / 3.0, cfl=0.4, limiter=1, amp=0.1):
    """grid-aligned CP Alfven wave along x (Eq. 10 as printed, with R2), Lx = 1, one wavelength"""
    x = cell_centres(nx, 1.0)
    ph = 2.0 * np.pi * x
    shp = (1, 1, nx)
    v = [np.zeros(shp), (amp * np.sin(ph)).reshape(shp), (amp * np.cos(ph)).reshape(shp)]
    Bc = [np.ones(shp), (amp * np.sin(ph)).reshape(shp), (amp * np.cos(ph)).reshape(shp)]
    faces = {"bx": np.ones((1, 1, nx + 1))}
    U = conserved_from_fields(np.ones(shp), v, Bc, np.full(shp, 0.1), gamma)
    return Workload(f"cp_alfven_1d_{nx}", nx, 1, 1, (1.0, 1.0 / nx, 1.0 / nx), gamma, cfl, limiter, 0, U,
                    join_faces(faces, nx, 1, 1), t_end=1.0)


# --------------------------------------------------------------------------- MHD blast (C3, C4)

def blast_3d(n=256, nsteps=50, seed=511, noise=1e-3, gamma=5.0 / 3.0, cfl=0.3, limiter=0, name=None,
             shape=None, p_in=10.0):
    nx, ny, nz = (n, n, n) if shape is None else shape
    L = (1.0, ny / nx, nz / nx)
    shp = (nz, ny, nx)
    xc, yc, zc = cell_centres(nx, L[0]), cell_centres(ny, L[1]), cell_centres(nz, L[2])
    r2 = ((xc[None, None, :] - 0.5 * L[0]) ** 2 + (yc[None, :, None] - 0.5 * L[1]) ** 2
          + (zc[:, None, None] - 0.5 * L[2]) ** 2)
    p = np.where(r2 < 0.1 ** 2, p_in, 0.1)
    u = counter_noise(seed, nx * ny * nz).reshape(shp)
    rho = 1.0 + noise * (2.0 * u - 1.0)
    b0 = 1.0 / np.sqrt(3.0)
    faces = {nm: np.full(s, b0) for nm, s in face_shapes(nx, ny, nz)}
    Bc = [np.full(shp, b0)] * 3
    zero = np.zeros(shp)
    U = conserved_from_fields(rho, [zero, zero, zero], Bc, p, gamma)
    return Workload(name or f"blast_3d_{nx}x{ny}x{nz}", nx, ny, nz, L, gamma, cfl, limiter, nsteps, U,
                    join_faces(faces, nx, ny, nz), seed=seed)


def blast_3d_planes(nx, ny, nz, k0, nzl, nblast=1, seed=511, noise=1e-3, gamma=5.0 / 3.0, p_in=10.0):
    """Planes [k0, k0 + nzl) of a blast problem in an nx x ny x nz box with cubic cells (Lx = 1), in the
    local layouts of a z slab (U[8][nzl][ny][nx]; bx, by with nzl planes, bz with nzl + 1): the weak-scaling
    workload of bench.py --gpus N, where the box grows along z with the number of GPUs and carries one
    blast of configs[3]'s recipe per slab-sized section (nblast of them, centred in their sections).  The
    noise is keyed by the GLOBAL linear cell index, so every rank generates exactly its part of one state."""
    L = (1.0, ny / nx, nz / nx)
    shp = (nzl, ny, nx)
    xc, yc = cell_centres(nx, L[0]), cell_centres(ny, L[1])
    zc = (np.arange(k0, k0 + nzl) + 0.5) * (L[2] / nz)
    sec = L[2] / nblast
    zrel = zc - (np.floor(zc / sec) + 0.5) * sec            # distance to the centre of the section
    r2 = (xc[None, None, :] - 0.5 * L[0]) ** 2 + (yc[None, :, None] - 0.5 * L[1]) ** 2 + zrel[:, None, None] ** 2
    p = np.where(r2 < 0.1 ** 2, p_in, 0.1)
    u = counter_noise(seed, nx * ny * nzl, start=k0 * nx * ny).reshape(shp)
    rho = 1.0 + noise * (2.0 * u - 1.0)
    b0 = 1.0 / np.sqrt(3.0)
    Bc = [np.full(shp, b0)] * 3
    zero = np.zeros(shp)
    U = conserved_from_fields(rho, [zero, zero, zero], Bc, p, gamma)
    Bl = np.full(nzl * ny * (nx + 1) + nzl * (ny + 1) * nx + (nzl + 1) * ny * nx, b0)
    return U, Bl, L


# --------------------------------------------------------------------------- generic small test problems

def random_smooth(nx, ny, nz, seed=1, gamma=5.0 / 3.0, cfl=0.3, limiter=0, amp=0.2, box=None):
    """smooth periodic random-phase state with divergence-free faces; ragged sizes welcome"""
    rng = np.random.default_rng(seed)
    L = box if box is not None else (1.0, ny / nx, nz / nx)
    shp = (nz, ny, nx)
    d = (L[0] / nx, L[1] / ny, L[2] / nz)
    xc, yc, zc = (cell_centres(n, l) for n, l in zip((nx, ny, nz), L))
    xf, yf, zf = (face_positions(n, l) for n, l in zip((nx, ny, nz), L))
    act = (nx > 1, ny > 1, nz > 1)

    def mode():
        k = [2 * np.pi * int(rng.integers(1, 3)) / L[a] if act[a] else 0.0 for a in range(3)]
        ph = rng.uniform(0, 2 * np.pi)
        return lambda xx, yy, zz: np.sin(k[0] * xx + k[1] * yy + k[2] * zz + ph)

    X = np.broadcast_to(xc[None, None, :], shp)
    Y = np.broadcast_to(yc[None, :, None], shp)
    Z = np.broadcast_to(zc[:, None, None], shp)
    rho = 1.0 + amp * mode()(X, Y, Z)
    p = 1.0 + amp * mode()(X, Y, Z)
    v = [amp * mode()(X, Y, Z) for _ in range(3)]
    fA = [mode() for _ in range(3)]
    B0 = rng.uniform(-0.5, 0.5, 3)
    Ax = amp * fA[0](xc[None, None, :], yf[None, :, None], zf[:, None, None]) * min(L) / (4.0 * np.pi)
    Ay = amp * fA[1](xf[None, None, :], yc[None, :, None], zf[:, None, None]) * min(L) / (4.0 * np.pi)
    Az = amp * fA[2](xf[None, None, :], yf[None, :, None], zc[:, None, None]) * min(L) / (4.0 * np.pi)
    faces = {}
    if act[0]:
        bx = np.full((nz, ny, nx + 1), B0[0])
        if act[1]:
            bx = bx + (Az[:, 1:, :] - Az[:, :-1, :]) / d[1]
        if act[2]:
            bx = bx - (Ay[1:, :, :] - Ay[:-1, :, :]) / d[2]
        faces["bx"] = bx
    if act[1]:
        by = np.full((nz, ny + 1, nx), B0[1])
        if act[2]:
            by = by + (Ax[1:, :, :] - Ax[:-1, :, :]) / d[2]
        if act[0]:
            by = by - (Az[:, :, 1:] - Az[:, :, :-1]) / d[0]
        faces["by"] = by
    if act[2]:
        bz = np.full((nz + 1, ny, nx), B0[2])
        if act[0]:
            bz = bz + (Ay[:, :, 1:] - Ay[:, :, :-1]) / d[0]
        if act[1]:
            bz = bz - (Ax[:, 1:, :] - Ax[:, :-1, :]) / d[1]
        faces["bz"] = bz
    Bc = [np.full(shp, B0[a]) + (0.0 if act[a] else amp * mode()(X, Y, Z)) for a in range(3)]
    Bc = cell_mean_of_faces(faces, nx, ny, nz, Bc)
    U = conserved_from_fields(rho, v, Bc, p, gamma)
    return Workload(f"random_smooth_{nx}x{ny}x{nz}", nx, ny, nz, tuple(L), gamma, cfl, limiter, 1, U,
                    join_faces(faces, nx, ny, nz), seed=seed)


# --------------------------------------------------------------------------- the BASELINE.json configs

def config(idx: int) -> Workload:
    """BASELINE.json configs[idx]"""
    if idx == 0:
        return orszag_tang_2d(128, nsteps=100, name="C0_orszag_tang_2d_128")
    if idx == 1:
        return cp_alfven_3d(64, name="C1_cp_alfven_3d_64x32x32")
    if idx == 2:
        return orszag_tang_2d(2048, nsteps=200, name="C2_orszag_tang_2d_2048")
    if idx == 3:
        return blast_3d(256, nsteps=50, name="C3_blast_3d_256")
    if idx == 4:
        return blast_3d(512, nsteps=20, name="C4_blast_3d_512")
    if idx == 5:    # not a BASELINE.json config: the paper's own 3D Orszag-Tang benchmark (section 4.1) at 256^3
        return orszag_tang_3d(256, noise=1e-3, name="P1_orszag_tang_3d_256")
    raise ValueError(idx)
