/*
 * pluto.h -- C-ABI boundary of libpluto_b200.so: the fp64 finite-volume ideal-MHD time step of
 * gPLUTO (arxiv 2511.20337) as hand-written CUDA kernels for sm_100a.
 *
 * The step (one call of pluto_step advances full RK2 steps) is, per RK stage:
 *   periodic ghost fill        (periodic boxes PAPER.md:254,360; pack/unpack Fig. 4)
 *   conservative -> primitive  (Eq. 7)
 *   PLM reconstruction of the primitives with a minmod / MC limiter (Eq. 6; reading R4)
 *   HLLD Riemann flux per sweep direction (Eq. 8; HLLD [56] PAPER.md:260; reading R5)
 *   flux-difference update     (Eq. 4; Fig. 2)
 *   constrained transport: upwind edge EMFs + face-B curl update (reading R6)
 * and once per step the RK2 combine (Eq. 5's increment form; reading R3) and the
 * CFL max-signal-speed reduction for dt (reading R8).  Readings R1..R20 are listed in DESIGN.md.
 * Beyond the north-star step: SSP-RK3 (Eq. 5 itself; PLUTO_OPT_RK_ORDER, reading R17) and WENO-Z
 * reconstruction ([51] named at PAPER.md:100,260; limiter PLUTO_WENOZ, reading R18).
 *
 * The EMF average of the paper's own runs, UCT-HLLD ([47] named at PAPER.md:271; reading R19): PLUTO_OPT_EMF.
 * The paper's other divergence control, GLM divergence cleaning ([43] named at PAPER.md:47,306,369; reading R20):
 * PLUTO_OPT_DIVB.
 * Beyond one GPU: the box cut into z slabs, one or more per process, with the ghost planes pulled out of
 * the neighbour slab's memory and one max for dt (section 3.4 "Multi GPU communication", PAPER.md:208-244,
 * Fig. 4; pluto_init_slabs and the calls below it).
 *
 * Everything is fp64.  One global context (the five north-star calls carry no handle).
 * All entry points return 0 (PLUTO_OK) or a negative error code; no exceptions, aborts or stdout.
 * There is NO CPU fallback: without a CUDA device every compute entry point returns PLUTO_ECUDA.
 *
 * Pointer arguments named U / Bface may be HOST or DEVICE pointers (the library asks the CUDA
 * runtime which); the caller owns them, the library copies in/out and never keeps them.
 *
 * Array layouts (doubles, SoA, i contiguous -- PAPER.md:154):
 *   U     : 8*nz*ny*nx, interior zones only, U[v][k][j][i]; v = 0 rho, 1-3 rho*v_{x,y,z},
 *           4-6 B_{x,y,z} (cell centred), 7 E   (component order of Eq. 2)
 *   Bface : [bx: nz*ny*(nx+1)] [by: nz*(ny+1)*nx] [bz: (nz+1)*ny*nx, only if nz > 1];
 *           face index 0 lies on the lower domain boundary; the last face of a family duplicates
 *           face 0 (periodic): ignored on input, written equal to face 0 on output.
 */
#ifndef PLUTO_B200_H
#define PLUTO_B200_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
    PLUTO_OK     =  0,
    PLUTO_EINVAL = -1,   /* bad argument */
    PLUTO_ESTATE = -2,   /* call order: not initialised / no state set */
    PLUTO_ECUDA  = -3,   /* CUDA runtime error or no device (see pluto_last_error) */
    PLUTO_EPHYS  = -4,   /* non-finite or non-positive density / pressure met during a step */
    PLUTO_ENOMEM = -5    /* device allocation failed or registered workspace too small */
};

/* reconstruction: PLM with the minmod / MC limiter (R4), or WENO-Z ([51]; R18; needs ghost >= 3) */
enum { PLUTO_MINMOD = 0, PLUTO_MC = 1, PLUTO_WENOZ = 2 };

/* pluto_init -- the mesh and the scheme (uniform Cartesian mesh of Eq. 4; periodic box,
 * PAPER.md:254,360; Gamma-law gas, Eq. 3).
 * Creates (or re-creates) the one global context for an nx x ny x nz periodic box of cubic cells with
 * Lx = 1 (override with pluto_set_box).  nx >= 2 and ny >= 2 (2D when nz == 1, 3D when nz >= 2); every
 * active extent >= ghost.  ghost = layers kept around the padded device arrays: >= 2 for PLM, >= 3 for
 * WENO-Z (R9), at most 16.  gamma > 1, cfl > 0 (R8), limiter = PLUTO_MINMOD | PLUTO_MC | PLUTO_WENOZ (R4, R18).
 * A call rejected with PLUTO_EINVAL (or PLUTO_ENOMEM for a registered workspace that is too small) leaves the
 * previous context untouched; once the arguments are accepted the previous context is released first.
 * Memory: allocates pluto_workspace_bytes(...) of device memory itself unless a workspace of at least that
 * size was registered with pluto_set_workspace (then the caller keeps ownership and must keep it alive
 * until pluto_finalize).  Errors: PLUTO_ECUDA (no device: there is no CPU fallback), PLUTO_EINVAL
 * (arguments), PLUTO_ENOMEM. */
int    pluto_init(int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter);

/* pluto_set_state -- the conserved state U of Eq. 2 and the staggered face field of the
 * constrained-transport method.
 * U: 8*nz*ny*nx doubles, Bface: the concatenated face arrays (layouts at the top of this file); each may
 * be a HOST or a DEVICE pointer, is only read, and is not kept after the call returns.  The cell-centred
 * B of every active dimension in U is ignored and replaced by the mean of its two faces (R7); E is taken
 * as given; the duplicate upper-boundary faces are ignored.  Resets the time to 0 and fills every ghost
 * zone (a1).  Errors: PLUTO_ESTATE (no pluto_init), PLUTO_EINVAL (NULL), PLUTO_ECUDA. */
int    pluto_set_state(const double *U, const double *Bface);

/* pluto_step -- nsteps full time steps of the semi-discrete scheme of Eq. 4 integrated
 * with SSP Runge-Kutta (Eq. 5; RK2 by default, R3): per stage ghost fill, cons->prim
 * (Eq. 7), reconstruction (Eq. 6), HLLD flux (Eq. 8), flux-difference update, CT; per step the CFL dt (R8)
 * computed on the device from the state at the start of the step.  Blocks until the work has completed on
 * the stream.  Errors: PLUTO_ESTATE (no state), PLUTO_EINVAL (nsteps < 0), PLUTO_EPHYS (a non-finite or
 * non-positive density / pressure was met: the state is then undefined, R13), PLUTO_ECUDA. */
int    pluto_step(int nsteps);

/* pluto_get_dt -- the CFL time step (R8; the paper does not print its rule): dt used by the most recent
 * step; before any step since pluto_set_state, the dt the next step will use (computed now).  Bit-identical
 * to an IEEE evaluation of dt = cfl / max_{zones, d} ((|v_d| + c_f,d) / dx_d) without contraction (R15).
 * NaN if there is no state. */
double pluto_get_dt(void);

/* pluto_get_state -- copy the state out in the layouts of pluto_set_state.  U, Bface: HOST or DEVICE
 * pointers to caller-owned memory of 8*nz*ny*nx and (sum of the face arrays) doubles; either may be
 * NULL.  U[4..6] of the active dimensions is the face mean (R7); the duplicate upper-boundary faces are
 * written equal to face 0.  Errors: PLUTO_ESTATE, PLUTO_ECUDA. */
int    pluto_get_state(double *U, double *Bface);

/* ---- extensions the five calls cannot express ---- */

int    pluto_set_box(double Lx, double Ly, double Lz);      /* cell sizes dx_d = L_d / n_d (R11) */
int    pluto_step_fixed_dt(int nsteps, double dt);          /* same step with dt imposed (R8: 1D pin, clipping) */
double pluto_get_time(void);                                /* sum of dt since set_state */
int    pluto_set_stream(void *cuda_stream);                 /* cudaStream_t to launch on (NULL: a stream of the library's own on the current device) */
/* Device memory one context needs (SSP-RK2; SSP-RK3 keeps a third state, which the library allocates itself on
 * first use unless the workspace was sized with pluto_workspace_bytes_slabs(..., rk_order = 3) and the
 * integrator was selected before pluto_init).  0 for sizes the library does not take. */
size_t pluto_workspace_bytes(int nx, int ny, int nz, int ghost);
/* caller-owned device memory (256-byte aligned) used by the next pluto_init / pluto_init_slabs; the
 * registration ends at pluto_finalize (the memory may then be freed); NULL: the library allocates */
int    pluto_set_workspace(void *dev, size_t bytes);
int    pluto_finalize(void);
const char *pluto_last_error(void);
int    pluto_device_count(void);                            /* 0 without a usable CUDA device */

/* ---- z-slab domain decomposition (section 3.4, Fig. 4) ----
 *
 * The nz planes of the box are cut into nslab slabs (the first nz % nslab slabs hold one plane more); every
 * slab has at least ghost + 1 planes.  This process holds slabs first .. first + count - 1:
 *   count == nslab : the whole box in one process, on one GPU.  Every other call of this header works
 *                    unchanged (pluto_step replays the whole step); results are bit-identical to
 *                    pluto_init for any nslab.
 *   count <  nslab : one process per GPU (count = 1, first = rank).  U / Bface of pluto_set_state and
 *                    pluto_get_state then cover only the planes held here ([bz] has local planes + 1), the
 *                    two outer neighbours are attached with pluto_attach_peer, and the step is driven in
 *                    phases so that the caller can place its collectives between them:
 *                        pluto_step_begin(0)            local part of the CFL max (a8)
 *                        [all-reduce MAX of the 8 bytes at pluto_dt_max_bits() over the processes]
 *                        pluto_step_stage(0, 0)         dt = cfl / max; ghost planes pulled from the peers; stage 1
 *                        [barrier: every process has finished its stage]
 *                        pluto_step_stage(1, 0) ...     one call per Runge-Kutta stage
 *                    The only data-path exchange is the ghost-plane pull inside the ghost-fill kernel (peer
 *                    loads over NVLink, no pack / unpack buffers: Fig. 4's Isend / Irecv pairs)
 *                    and the one max for dt.
 * Errors: as pluto_init; PLUTO_EINVAL for a slab thinner than ghost + 1 planes or nz < 2. */
int    pluto_init_slabs(int nslab, int first, int count, int nx, int ny, int nz, int ghost,
                        double gamma, double cfl, int limiter);
size_t pluto_workspace_bytes_slabs(int nslab, int first, int count, int nx, int ny, int nz, int ghost, int rk_order);
/* planes of slab `slab` when nz planes are cut into nslab slabs: first plane and count (no device needed) */
int    pluto_slab_planes(int nz, int nslab, int slab, int *k0, int *planes);
/* first global plane and number of planes this process holds */
int    pluto_local_planes(int *k0, int *nz_local);
/* The memory of the lowest (side 0) or highest (side 1) slab held here, for the neighbour process to attach:
 * a 64-byte CUDA IPC handle (ipc_handle64, may be NULL; only for memory the library allocated itself), the
 * device pointer (device_ptr, for a neighbour in the same process or with peer access), the array stride
 * in doubles and the number of interior planes.  Any output pointer may be NULL. */
int    pluto_export_slab(int side, void *ipc_handle64, void **device_ptr, long long *array_stride, int *planes);
/* Attach the slab below (side 0) or above (side 1) the planes held here: either its IPC handle (opened with
 * peer access enabled; closed at pluto_finalize) or a device pointer valid in this process. */
int    pluto_attach_peer(int side, const void *ipc_handle64, void *device_ptr, long long array_stride, int planes);
/* fill every ghost zone of the current state (a1) once all processes have set their state */
int    pluto_fill_ghosts(void);
/* Phases of one step (see above).  fixed_dt > 0: impose dt (no reduction); pass fixed = 1 to pluto_step_stage.
 * Nothing here waits for the device: the calls enqueue on the stream; pluto_sync reports errors. */
int    pluto_step_begin(double fixed_dt);
void  *pluto_dt_max_bits(void);        /* DEVICE pointer to the running max of (|v_d| + c_f,d)/dx_d as the bit
                                          pattern of a positive double (an order-preserving unsigned 64-bit integer) */
int    pluto_step_stage(int stage, int fixed);

/* Enqueue nsteps steps without waiting (no error check, no host synchronisation); used for timing
 * with CUDA events on the stream given to pluto_set_stream.  pluto_sync waits and returns
 * PLUTO_EPHYS / PLUTO_ECUDA like pluto_step. */
int    pluto_step_async(int nsteps);
int    pluto_sync(void);

/* Tuning switches: opt = PLUTO_OPT_*, returns the previous value or PLUTO_EINVAL. */
enum {
    PLUTO_OPT_GRAPH = 1,   /* 1 (default): replay one captured CUDA graph per step; 0: plain launches */
    PLUTO_OPT_FUSE_XY = 2, /* 1 (default): x and y sweeps fused in one kernel; 0: one kernel per direction */
    PLUTO_OPT_CT_TMA = 3,  /* 1 (default): CT operands staged by TMA (cp.async.bulk.tensor); 0: per-thread loads */
    PLUTO_OPT_RK_ORDER = 4,/* 2 (default): SSP-RK2 (north star, reading R3); 3: SSP-RK3 of Eq. 5 (R17) */
    PLUTO_OPT_DIVB = 5,    /* divergence control of the NEXT pluto_init: PLUTO_DIVB_CT (default) or PLUTO_DIVB_GLM */
    PLUTO_OPT_EMF = 6      /* EMF average of the constrained-transport step: PLUTO_EMF_CONTACT (default) or PLUTO_EMF_UCT_HLLD */
};
/* Divergence control: constrained transport (the north-star path), or the GLM
 * divergence cleaning of [43] (reading R20 in DESIGN.md): cell-centred B, one more scalar
 * psi, no face fields.  With PLUTO_DIVB_GLM: PLM only, one domain; pluto_set_state reads the cell-centred field
 * from U[4..6] and ignores Bface (may be NULL), psi starts at zero; pluto_get_state writes U only. */
enum { PLUTO_DIVB_CT = 0, PLUTO_DIVB_GLM = 1 };
/* EMF average of the constrained-transport step: PLUTO_EMF_CONTACT, the upwind-by-contact-mode
 * rule with the continuous weight (reading R6; the north-star path, fused x+y sweep, TMA-staged CT kernel), or
 * PLUTO_EMF_UCT_HLLD, the UCT-HLLD average of [47] that the paper's runs use (reference entry :640;
 * reading R19 in DESIGN.md: the interface coefficients are the linear decomposition of the HLLD induction flux,
 * the edge value is composed from them with the run's reconstruction).  May be switched at any time outside a
 * step; the first step in UCT-HLLD mode allocates six more work arrays per slab with cudaMalloc (freed by
 * pluto_finalize).  Ignored by the GLM variant. */
enum { PLUTO_EMF_CONTACT = 0, PLUTO_EMF_UCT_HLLD = 1 };
int    pluto_set_psi(const double *psi);      /* [nz][ny][nx], host or device; GLM variant only */
int    pluto_get_psi(double *psi);
int    pluto_set_option(int opt, int value);

/* pluto_cfl_dt_noalloc -- the CFL time step (reading R8; the same rule as pluto_get_dt) of a state the CALLER
 * holds, computed without the library allocating anything: no context, no pluto_init, no cudaMalloc / cudaFree,
 * no allocating library routine.
 *
 * Who needs it: a host code that gives all device memory to its own pool when it starts (an AMR framework's
 * arena, a caching allocator run close to the full HBM) cannot rely on a library-side cudaMalloc succeeding;
 * and a caller inside a latency-critical loop cannot pay for the device-wide synchronisation cudaMalloc and
 * cudaFree bring.  pluto_init / pluto_get_dt allocate (or need a registered workspace of many arrays); this
 * call needs only the caller's own input and output.
 *
 *   U_dev   : DEVICE pointer, 8*nz*ny*nx doubles in the layout of pluto_get_state's U (interior zones only,
 *             cell-centred B in U[4..6]); only read
 *   nx,ny,nz: zones (nx >= 2, ny >= 2, nz >= 1; 2D when nz == 1); Lx,Ly,Lz: box lengths, dx_d = L_d / n_d (R11)
 *   out_dev : DEVICE pointer to 3 doubles the caller owns: out[0] = dt = cfl / max, out[1] = the maximum of
 *             (|v_d| + c_f,d) / dx_d over zones and active d, out[2] = 1.0 if a zone with non-positive or
 *             non-finite density / pressure was met (R13), else 0.0
 *   cuda_stream : cudaStream_t to enqueue on (NULL: the default stream).  The call only enqueues (one memset
 *             and two kernels) and does not wait: synchronise the stream before reading out_dev.
 * For the same state, box, gamma and cfl, out[0] is bit-identical to pluto_get_dt() (R15).
 *
 * The scratch in between (one partial maximum per row of nx zones, plus a flag word) is a fixed array inside
 * the library's device image: PLUTO_NOALLOC_SCRATCH_BYTES (1 MiB + 256 B) on every GPU that loads the library,
 * held until the process exits.  Hence the limit ny * nz <= PLUTO_NOALLOC_MAX_ROWS (256^3 is 65 536 rows,
 * 2048^2 is 2 048): larger boxes are refused with PLUTO_ENOMEM and a message in pluto_last_error; nothing is
 * launched.  Every call on a device uses the same array and finds the previous call's contents in it: the call
 * clears the flag word itself and overwrites every row maximum before reading it, so consecutive calls on one
 * stream are independent -- but two calls that may run at the same time on one GPU (different streams, or
 * different host threads) race on it and must be ordered by the caller.
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 * current) and keeps it; make that first call outside any stream capture.
 * Errors: PLUTO_EINVAL (NULL pointer, sizes, lengths, gamma, cfl), PLUTO_ENOMEM (more rows than the scratch
 * holds), PLUTO_ECUDA (no device -- there is no CPU fallback -- or a CUDA runtime error). */
#define PLUTO_NOALLOC_MAX_ROWS      131072
#define PLUTO_NOALLOC_SCRATCH_BYTES ((PLUTO_NOALLOC_MAX_ROWS + 32) * 8)
int    pluto_cfl_dt_noalloc(const double *U_dev, int nx, int ny, int nz, double Lx, double Ly, double Lz,
                            double gamma, double cfl, double *out_dev, void *cuda_stream);

/* Test, timing and profiling entry points (pluto_debug_euler, pluto_profile*, pluto_launch_count,
 * pluto_graph_captures, pluto_probe_fp64_gflops) are exported by the same library and declared in pluto_debug.h. */

#ifdef __cplusplus
}
#endif
#endif
