/*
 * pluto_debug.h -- entry points of libpluto_b200.so that serve the tests and bench.py, not a production caller:
 * per-kernel parity (pluto_debug_euler), launch / graph-capture counters, per-kernel CUDA-event timing and the
 * fp64 peak probe behind bench.py's roofline.  The product ABI (the five north-star calls, their
 * extensions, the z-slab calls and the options) is include/pluto.h; conventions (error codes, layouts, host or
 * device pointers) are the ones stated there.
 */
#ifndef PLUTO_B200_DEBUG_H
#define PLUTO_B200_DEBUG_H
#include "pluto.h"
#ifdef __cplusplus
extern "C" {
#endif

/* Number of kernel launches enqueued by this library since pluto_init (for bench.py's gpu_launches). */
long long pluto_launch_count(void);

/* Per-kernel device timing with CUDA events on the launching stream (for bench.py's roofline).
 * pluto_profile(1) starts (plain launches, every launch bracketed by an event pair), pluto_profile(0)
 * stops.  pluto_profile_get returns the accumulated time and launch count of kernel class `kernel`
 * (0 <= kernel, pluto_kernel_name(kernel) != NULL). */
int    pluto_profile(int on);
int    pluto_profile_get(int kernel, double *total_ms, long long *launches);
const char *pluto_kernel_name(int kernel);

/* Measured fp64 FMA throughput of the device in GFLOP/s (2 flops per DFMA): a register-resident
 * DFMA loop on every SM, timed with CUDA events.  The denominator of the "alu" roofline. */
double pluto_probe_fp64_gflops(void);

/* Number of CUDA graph captures (capture + instantiate of one whole step) since the library was loaded.  A run of
 * pluto_step / pluto_step_async calls with unchanged options captures once per dt mode; a test uses the counter
 * to check that nothing re-captures per step. */
long long pluto_graph_captures(void);

/* One Euler stage S -> S + L(S) from the CURRENT state with the given dt, for per-kernel parity
 * tests; the state is not advanced.  Any pointer may be NULL (host or device pointers).
 *   U1, Bf1 : layouts of U / Bface
 *   W       : [3][nz][ny][nx] upwind weight on the LOWER d-face of each cell (R6)
 *   Fem     : [3][2][nz][ny][nx] the two induction fluxes kept for CT on that face:
 *             d = x: (F_x[B_y], F_x[B_z]);  d = y: (F_y[B_z], F_y[B_x]);  d = z: (F_z[B_x], F_z[B_y])
 *   Eedge   : [3][nz][ny][nx] Ex at (i, j-1/2, k-1/2), Ey at (i-1/2, j, k-1/2), Ez at (i-1/2, j-1/2, k)
 * entries of inactive directions are zero.  In UCT-HLLD mode (PLUTO_OPT_EMF) the scheme keeps no W and no Fem:
 * a non-NULL W or Fem is refused with PLUTO_ESTATE. */
int    pluto_debug_euler(double dt, double *U1, double *Bf1, double *W, double *Fem, double *Eedge);

#ifdef __cplusplus
}
#endif
#endif
