/*
 * oracle.h -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU implementation (C99, fp64, no FMA
 * contraction) of the finite-volume ideal-MHD time step whose CUDA version
 * lives in paper_2511_20337_b200/csrc.  It shares no code with the CUDA path
 * and must never be linked, imported or executed by it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may use anything under oracle/.
 *
 * Citations are "PAPER.md:<line>" of arxiv 2511.20337 plus the equation /
 * section.  Where the paper names a method without printing its formulas the
 * reading taken is listed in DESIGN.md ("Readings R1..R16") and cited as R<n>.
 *
 * Layouts (all doubles, SoA, i fastest -- PAPER.md:154):
 *   U     : 8*nz*ny*nx, U[v][k][j][i], v = 0 rho, 1-3 rho*v, 4-6 B (cell), 7 E
 *           (component order of Eq. 2).
 *   Bface : [bx: nz*ny*(nx+1)] [by: nz*(ny+1)*nx] [bz: (nz+1)*ny*nx];
 *           a family is present only if its direction is active (n_d > 1);
 *           face index 0 is the lower domain boundary, the last face duplicates
 *           face 0 (periodic boxes).
 */
#ifndef ORACLE_H
#define ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_ESTATE = -2, ORACLE_EPHYS = -4, ORACLE_ENOMEM = -5 };

/* ---- the five calls of the boundary + extensions (same meaning as include/pluto.h) ---- */
int    oracle_init(int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter);
int    oracle_set_box(double Lx, double Ly, double Lz);
int    oracle_set_state(const double *U, const double *Bface);
int    oracle_step(int nsteps);
int    oracle_step_fixed_dt(int nsteps, double dt);
double oracle_get_dt(void);
double oracle_get_time(void);
int    oracle_get_state(double *U, double *Bface);
int    oracle_finalize(void);
int    oracle_set_integrator(int order); /* after oracle_init: 2 = SSP-RK2 (default, R3), 3 = SSP-RK3 of Eq. 5 (R17) */
int    oracle_set_threads(int n);      /* OpenMP threads (results do not depend on it) */
int    oracle_get_threads(void);

/* ---- GLM divergence cleaning ([43] PAPER.md:636; reading R20 in oracle.c) ----
 * oracle_set_divb(1) after oracle_init switches to the cell-centred-B variant: U[4..6] is the field, Bface is
 * ignored (may be NULL), psi starts at zero (oracle_set_psi overrides it).  0 = constrained transport (default). */
int    oracle_set_divb(int mode);
int    oracle_set_psi(const double *psi);       /* [nz][ny][nx] */
int    oracle_get_psi(double *psi);
/* exact interface state of the (B_n, psi) subsystem with the waves -c_h, +c_h */
void   oracle_glm_interface(double BnL, double BnR, double psiL, double psiR, double ch, double *Bm, double *psim);

/* ---- pieces, exposed so that tests can pin each one separately ---- */

/* Eq. 7: U[8] -> V[8] = (rho, vx, vy, vz, Bx, By, Bz, p). returns 0, or ORACLE_EPHYS */
int    oracle_cons2prim(const double U[8], double gamma, double V[8]);
/* Eq. 3: V[8] -> U[8] */
void   oracle_prim2cons(const double V[8], double gamma, double U[8]);
/* fast magnetosonic speed along the direction whose field component is Bn (R5/R8) */
double oracle_fast_speed(double rho, double p, double Bn, double Bt1, double Bt2, double gamma);
/* limited slope from the two one-sided differences (R4); limiter 0 = minmod, 1 = MC */
double oracle_plm_slope(double dm, double dp, int limiter);
/* WENO-Z value at the upper face of the centre cell of a five-cell stencil ([51] named at PAPER.md:100; R18);
   reconstruction id 2 of oracle_init's `limiter` argument */
double oracle_wenoz(const double v[5]);
/* physical flux of Eq. 2 in the rotated frame.
   V = (rho, u, v, w, By, Bz, p), Bn normal field. F = (rho, mn, mt1, mt2, 0, Bt1, Bt2, E) */
void   oracle_physical_flux(const double V[7], double Bn, double gamma, double F[8]);
/* HLLD flux (R5) in the rotated frame + continuous upwind weight w (R6).
   dbg (may be NULL) receives 72 doubles:
   [0]SL [1]SR [2]SM [3]pT* [4]S*L [5]S*R [6]region(0..5) [7]unused
   [8..15]UL [16..23]UR [24..31]U*L [32..39]U*R [40..47]U**L [48..55]U**R [56..63]FL [64..71]FR
   (when the fan is one-sided, the star entries are not filled) */
int    oracle_hlld(const double VL[7], const double VR[7], double Bn, double gamma,
                   double F[8], double *w, double *dbg);

/* the same, also returning uct[5] = a^L, d^L, d^R and the two transverse velocities a^L v_t^L + a^R v_t^R of the
   UCT-HLLD EMF average ([47] named at PAPER.md:271; reading R19, formulas in oracle.c) */
int    oracle_hlld_uct(const double VL[7], const double VR[7], double Bn, double gamma,
                       double F[8], double *w, double *dbg, double *uct);
/* after oracle_init: EMF average of the constrained-transport step: 0 = upwind by the contact mode with the
   continuous weight (R6, default), 1 = UCT-HLLD (R19) */
int    oracle_set_emf(int mode);

/* One Euler stage S -> S + L(S) (R1, Eq. 4) from the CURRENT state with the given
   dt; the state is not modified.  Any output pointer may be NULL.
     U1, Bf1 : same layouts as U / Bface
     F       : [3][8][nz][ny][nx] lab-frame flux through the LOWER d-face of each cell
     W       : [3][nz][ny][nx]    upwind weight on that face
     Eedge   : [3][nz][ny][nx]    Ex at (i, j-1/2, k-1/2), Ey at (i-1/2, j, k-1/2), Ez at (i-1/2, j-1/2, k)
   entries of inactive directions are zero. */
int    oracle_debug_euler(double dt, double *U1, double *Bf1, double *F, double *W, double *Eedge);

#ifdef __cplusplus
}
#endif
#endif
