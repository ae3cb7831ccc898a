/*
 * oracle.c -- TEST INFRASTRUCTURE ONLY (see oracle.h).
 *
 * Step-by-step CPU restatement of the finite-volume ideal-MHD time step of
 * arxiv 2511.20337 (gPLUTO): cons->prim (Eq. 7), PLM reconstruction on
 * primitives (Eq. 6 + R4), HLLD Riemann flux (Eq. 8, [56], R5), flux-difference
 * update (Eq. 4, Fig. 2), constrained transport with an upwind edge-EMF average
 * (R6), SSP-RK2 in the increment form of Eq. 5 (R3), CFL time step
 * (R8) on periodic boxes.  No ghost zones: every neighbour
 * index is taken modulo n.  No blocking, fusion or reordering; loops are in the
 * order the text states.  Build: gcc -O2 -std=c99 -ffp-contract=off [-fopenmp].
 *
 * PARITY PINS: every function here is pinned by tests/test_oracle_*.py against
 * closed forms, invariants and textbook special cases, EXCEPT the absolute field
 * values of the Orszag-Tang and blast runs, which the paper does not print:
 * "parity unpinned" for those values (only invariants pin them).
 */
#include "oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* upwind-weight sharpness of R6: |mass flux| >= THETA * f_ref is fully upwinded */
#define THETA 1e-3
/* degeneracy guard of the HLLD star-state denominator (R5) */
#define DEGEN 1e-8

typedef struct {
    int init;
    int n[3];            /* nx, ny, nz */
    int act[3];          /* direction active (n_d > 1) */
    double L[3], dx[3];
    double gamma, cfl;
    int limiter;
    size_t N;
    double *U;           /* [8][N] */
    double *b[3];        /* face fields, [N] each, index c = lower d-face of cell c */
    /* stage buffers */
    double *U1, *U2, *b1[3], *b2[3];
    /* work */
    double *V, *F, *W, *Eg, *Ec;
    /* EMF average: 0 = upwind by the contact mode with the continuous weight (R6, default),
       1 = UCT-HLLD (R19); its face data [3][5][N]: a^L, d^L, d^R, transverse velocities t1, t2 */
    int emf;
    double *Uct;
    double time, dt_last;
    int stepped;
    int rk_order;          /* 2 (or 0: default) = SSP-RK2, 3 = SSP-RK3 */
    int err;
    int threads;
    /* divergence control: 0 = constrained transport (default), 1 = GLM divergence cleaning (R20) */
    int divb;
    double *psi, *psi1, *psi2;   /* the cleaning scalar of the GLM variant, [N] each */
    double *Fpsi;                /* its flux through the lower d-face, [3][N] */
} ctx_t;

static ctx_t g;

/* ------------------------------------------------------------------ helpers */

static int wrap(int i, int n) { i %= n; return i < 0 ? i + n : i; }

static size_t cidx(int i, int j, int k) {
    return ((size_t)wrap(k, g.n[2]) * g.n[1] + wrap(j, g.n[1])) * g.n[0] + wrap(i, g.n[0]);
}

/* index of the cell shifted by s along direction d from (i,j,k) */
static size_t shift(int i, int j, int k, int d, int s) {
    int q[3] = { i, j, k };
    q[d] += s;
    return cidx(q[0], q[1], q[2]);
}

static void c2ijk(size_t c, int *i, int *j, int *k) {
    *i = (int)(c % g.n[0]);
    *j = (int)((c / g.n[0]) % g.n[1]);
    *k = (int)(c / ((size_t)g.n[0] * g.n[1]));
}

/* ------------------------------------------------------------------ pieces */

/* Eq. 7 */
int oracle_cons2prim(const double U[8], double gamma, double V[8])
{
    double rho = U[0];
    double vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
    double p = (gamma - 1.0) * (U[7] - 0.5 * (U[1] * vx + U[2] * vy + U[3] * vz)
                                     - 0.5 * (U[4] * U[4] + U[5] * U[5] + U[6] * U[6]));
    V[0] = rho; V[1] = vx; V[2] = vy; V[3] = vz;
    V[4] = U[4]; V[5] = U[5]; V[6] = U[6]; V[7] = p;
    if (!(rho > 0.0) || !(p > 0.0) || !isfinite(rho) || !isfinite(p)) return ORACLE_EPHYS;
    return ORACLE_OK;
}

/* Eq. 3 */
void oracle_prim2cons(const double V[8], double gamma, double U[8])
{
    U[0] = V[0];
    U[1] = V[0] * V[1]; U[2] = V[0] * V[2]; U[3] = V[0] * V[3];
    U[4] = V[4]; U[5] = V[5]; U[6] = V[6];
    U[7] = V[7] / (gamma - 1.0) + 0.5 * V[0] * (V[1] * V[1] + V[2] * V[2] + V[3] * V[3])
         + 0.5 * (V[4] * V[4] + V[5] * V[5] + V[6] * V[6]);
}

/* fast magnetosonic speed (R5): c_f^2 = ( s + sqrt(s^2 - 4 a^2 bn^2) ) / 2, s = a^2 + b^2 */
double oracle_fast_speed(double rho, double p, double Bn, double Bt1, double Bt2, double gamma)
{
    double a2  = gamma * p / rho;
    double b2  = (Bn * Bn + Bt1 * Bt1 + Bt2 * Bt2) / rho;
    double bn2 = Bn * Bn / rho;
    double s   = a2 + b2;
    double disc = s * s - 4.0 * a2 * bn2;
    if (disc < 0.0) disc = 0.0;
    return sqrt(0.5 * (s + sqrt(disc)));
}

/* R4: minmod / monotonised-central limited slope from dm = q_c - q_{c-1}, dp = q_{c+1} - q_c */
double oracle_plm_slope(double dm, double dp, int limiter)
{
    if (!(dm * dp > 0.0)) return 0.0;
    if (limiter == 0) return (fabs(dm) < fabs(dp)) ? dm : dp;
    {
        double sum = dm + dp;
        double m2 = 2.0 * fmin(fabs(dm), fabs(dp));
        double c2 = 0.5 * fabs(sum);
        double mag = fmin(m2, c2);
        return sum > 0.0 ? mag : -mag;
    }
}

/* WENO-Z reconstruction of [51] (Borges, Carmona, Costa & Don 2008; named at PAPER.md:100,260; reading R18):
   value at the UPPER face of the centre cell v[2] from the five-cell stencil v[0..4].
   Candidate third-order values q_k, smoothness indicators beta_k (Jiang-Shu), global indicator
   tau5 = |beta_0 - beta_2|, weights alpha_k = d_k (1 + tau5 / (beta_k + eps)), d = (1/10, 6/10, 3/10),
   eps = 1e-40, power 1.  The value at the LOWER face is the same routine on the mirrored stencil. */
double oracle_wenoz(const double v[5])
{
    const double eps = 1e-40;
    double q0 = (2.0 * v[0] - 7.0 * v[1] + 11.0 * v[2]) / 6.0;
    double q1 = (-v[1] + 5.0 * v[2] + 2.0 * v[3]) / 6.0;
    double q2 = (2.0 * v[2] + 5.0 * v[3] - v[4]) / 6.0;
    double a0 = v[0] - 2.0 * v[1] + v[2], b0 = v[0] - 4.0 * v[1] + 3.0 * v[2];
    double a1 = v[1] - 2.0 * v[2] + v[3], b1 = v[1] - v[3];
    double a2 = v[2] - 2.0 * v[3] + v[4], b2 = 3.0 * v[2] - 4.0 * v[3] + v[4];
    double be0 = 13.0 / 12.0 * a0 * a0 + 0.25 * b0 * b0;
    double be1 = 13.0 / 12.0 * a1 * a1 + 0.25 * b1 * b1;
    double be2 = 13.0 / 12.0 * a2 * a2 + 0.25 * b2 * b2;
    double tau = fabs(be0 - be2);
    double al0 = 0.1 * (1.0 + tau / (be0 + eps));
    double al1 = 0.6 * (1.0 + tau / (be1 + eps));
    double al2 = 0.3 * (1.0 + tau / (be2 + eps));
    return (al0 * q0 + al1 * q1 + al2 * q2) / (al0 + al1 + al2);
}

/* rotated-frame conserved vector (rho, mn, mt1, mt2, Bn, Bt1, Bt2, E) from V = (rho,u,v,w,By,Bz,p) */
static void rot_cons(const double V[7], double Bn, double gamma, double U[8])
{
    double rho = V[0], u = V[1], v = V[2], w = V[3], By = V[4], Bz = V[5], p = V[6];
    U[0] = rho; U[1] = rho * u; U[2] = rho * v; U[3] = rho * w;
    U[4] = Bn; U[5] = By; U[6] = Bz;
    U[7] = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * (Bn * Bn + By * By + Bz * Bz);
}

/* Eq. 2, normal component of T in the rotated frame */
void oracle_physical_flux(const double V[7], double Bn, double gamma, double F[8])
{
    double rho = V[0], u = V[1], v = V[2], w = V[3], By = V[4], Bz = V[5], p = V[6];
    double B2 = Bn * Bn + By * By + Bz * Bz;
    double pT = p + 0.5 * B2;
    double vB = u * Bn + v * By + w * Bz;
    double E  = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w) + 0.5 * B2;
    F[0] = rho * u;
    F[1] = rho * u * u + pT - Bn * Bn;
    F[2] = rho * u * v - Bn * By;
    F[3] = rho * u * w - Bn * Bz;
    F[4] = 0.0;
    F[5] = By * u - Bn * v;
    F[6] = Bz * u - Bn * w;
    F[7] = (E + pT) * u - Bn * vB;
}

/* HLLD (Miyoshi & Kusano, [56] PAPER.md:649) as read in R5, plus the weight of R6 */
int oracle_hlld(const double VL[7], const double VR[7], double Bn, double gamma,
                double F[8], double *wout, double *dbg)
{
    return oracle_hlld_uct(VL, VR, Bn, gamma, F, wout, dbg, NULL);
}

/* The same solver, also returning (uct != NULL) what the UCT-HLLD EMF average of [47] (named at PAPER.md:271,
   reference entry :640; reading R19) takes from every interface.  For fixed wave speeds the HLLD flux of a
   transverse field component B_t is LINEAR in (v_t^L, v_t^R, B_t^L, B_t^R); writing it as

       F[B_t] = a^L (u B_t)^L + a^R (u B_t)^R - (d^R B_t^R - d^L B_t^L) - B_n (a^L v_t^L + a^R v_t^R)

   fixes the four coefficients uniquely (a^L + a^R = 1).  With lambda^L = S_L, lambda^R = S_R, the Alfven speeds
   lambda^*L = S*_L, lambda^*R = S*_R and lambda_c = S_M:

       chi^s = (u^s - lambda_c)(lambda^s - lambda_c) / (lambda^*s + lambda^s - 2 lambda_c)
       nu^s  = (lambda^*s + lambda^s) / (|lambda^*s| + |lambda^s|)
       nu^*  = (lambda^*R + lambda^*L) / (|lambda^*R| + |lambda^*L|)      (0 when both Alfven speeds vanish)
       a^L = (1 + nu^*)/2,  a^R = (1 - nu^*)/2
       d^s = (nu^s - nu^*) chi^s / 2 + (|lambda^*s| - nu^* lambda^*s) / 2

   (one-sided fans: a = 1 on the upwind side, d^L = d^R = 0).  tests/test_oracle_uct.py checks the identity above
   against the flux this routine returns, region by region.
   uct[5] = a^L, d^L, d^R, a^L v^L + a^R v^R (first transverse velocity), a^L w^L + a^R w^R (second). */
int oracle_hlld_uct(const double VL[7], const double VR[7], double Bn, double gamma,
                    double F[8], double *wout, double *dbg, double *uct)
{
    const double *Va[2] = { VL, VR };
    double U[2][8], Fp[2][8], pT[2], vB[2], cf[2], S[2];
    double Us[2][8], Uss[2][8], vBs[2], Sa[2];
    double SM, pTs, wgt, fref;
    int a, v, region;
    double Bx = Bn;

    for (a = 0; a < 2; a++) {
        const double *q = Va[a];
        double B2 = Bx * Bx + q[4] * q[4] + q[5] * q[5];
        pT[a] = q[6] + 0.5 * B2;
        vB[a] = q[1] * Bx + q[2] * q[4] + q[3] * q[5];
        rot_cons(q, Bx, gamma, U[a]);
        oracle_physical_flux(q, Bx, gamma, Fp[a]);
        cf[a] = oracle_fast_speed(q[0], q[6], Bx, q[4], q[5], gamma);
    }
    /* outer speeds (R5) */
    {
        double cmax = fmax(cf[0], cf[1]);
        S[0] = fmin(VL[1], VR[1]) - cmax;
        S[1] = fmax(VL[1], VR[1]) + cmax;
    }
    fref = 0.25 * (VL[0] + VR[0]) * (S[1] - S[0]);

    if (dbg) {
        memset(dbg, 0, 72 * sizeof(double));
        dbg[0] = S[0]; dbg[1] = S[1];
        for (v = 0; v < 8; v++) { dbg[8 + v] = U[0][v]; dbg[16 + v] = U[1][v]; dbg[56 + v] = Fp[0][v]; dbg[64 + v] = Fp[1][v]; }
    }

    if (S[0] >= 0.0) {
        for (v = 0; v < 8; v++) F[v] = Fp[0][v];
        region = 0;
        if (uct) { uct[0] = 1.0; uct[1] = 0.0; uct[2] = 0.0; uct[3] = VL[2]; uct[4] = VL[3]; }
    } else if (S[1] <= 0.0) {
        for (v = 0; v < 8; v++) F[v] = Fp[1][v];
        region = 5;
        if (uct) { uct[0] = 0.0; uct[1] = 0.0; uct[2] = 0.0; uct[3] = VR[2]; uct[4] = VR[3]; }
    } else {
        double aL = VL[0] * (S[0] - VL[1]);
        double aR = VR[0] * (S[1] - VR[1]);
        double am[2];
        am[0] = aL; am[1] = aR;
        SM  = (aR * VR[1] - aL * VL[1] - pT[1] + pT[0]) / (aR - aL);
        pTs = (aR * pT[0] - aL * pT[1] + aL * aR * (VR[1] - VL[1])) / (aR - aL);

        for (a = 0; a < 2; a++) {
            const double *q = Va[a];
            double rhos = am[a] / (S[a] - SM);
            double D = am[a] * (S[a] - SM) - Bx * Bx;
            double vs, ws, Bys, Bzs, Es;
            if (fabs(D) <= DEGEN * pTs) {
                vs = q[2]; ws = q[3]; Bys = q[4]; Bzs = q[5];
            } else {
                double num = am[a] * (S[a] - q[1]) - Bx * Bx;
                vs  = q[2] - Bx * q[4] * (SM - q[1]) / D;
                ws  = q[3] - Bx * q[5] * (SM - q[1]) / D;
                Bys = q[4] * num / D;
                Bzs = q[5] * num / D;
            }
            vBs[a] = SM * Bx + vs * Bys + ws * Bzs;
            Es = ((S[a] - q[1]) * U[a][7] - pT[a] * q[1] + pTs * SM + Bx * (vB[a] - vBs[a])) / (S[a] - SM);
            Us[a][0] = rhos; Us[a][1] = rhos * SM; Us[a][2] = rhos * vs; Us[a][3] = rhos * ws;
            Us[a][4] = Bx;   Us[a][5] = Bys;       Us[a][6] = Bzs;       Us[a][7] = Es;
        }
        /* Alfven speeds */
        {
            double rL = sqrt(Us[0][0]), rR = sqrt(Us[1][0]);
            double sig = (double)((Bx > 0.0) - (Bx < 0.0));
            double R = rL + rR;
            double vsL = Us[0][2] / Us[0][0], wsL = Us[0][3] / Us[0][0];
            double vsR = Us[1][2] / Us[1][0], wsR = Us[1][3] / Us[1][0];
            double vss, wss, Byss, Bzss, vBss;
            Sa[0] = SM - fabs(Bx) / rL;
            Sa[1] = SM + fabs(Bx) / rR;
            vss  = (rL * vsL + rR * vsR + sig * (Us[1][5] - Us[0][5])) / R;
            wss  = (rL * wsL + rR * wsR + sig * (Us[1][6] - Us[0][6])) / R;
            Byss = (rL * Us[1][5] + rR * Us[0][5] + sig * rL * rR * (vsR - vsL)) / R;
            Bzss = (rL * Us[1][6] + rR * Us[0][6] + sig * rL * rR * (wsR - wsL)) / R;
            vBss = SM * Bx + vss * Byss + wss * Bzss;
            for (a = 0; a < 2; a++) {
                double r = a == 0 ? rL : rR;
                double sg = a == 0 ? -sig : sig;
                Uss[a][0] = Us[a][0]; Uss[a][1] = Us[a][0] * SM;
                Uss[a][2] = Us[a][0] * vss; Uss[a][3] = Us[a][0] * wss;
                Uss[a][4] = Bx; Uss[a][5] = Byss; Uss[a][6] = Bzss;
                Uss[a][7] = Us[a][7] + sg * r * (vBs[a] - vBss);
            }
        }
        if (Sa[0] >= 0.0) {
            for (v = 0; v < 8; v++) F[v] = Fp[0][v] + S[0] * (Us[0][v] - U[0][v]);
            region = 1;
        } else if (SM >= 0.0) {
            for (v = 0; v < 8; v++)
                F[v] = Fp[0][v] + Sa[0] * Uss[0][v] - (Sa[0] - S[0]) * Us[0][v] - S[0] * U[0][v];
            region = 2;
        } else if (Sa[1] > 0.0) {
            for (v = 0; v < 8; v++)
                F[v] = Fp[1][v] + Sa[1] * Uss[1][v] - (Sa[1] - S[1]) * Us[1][v] - S[1] * U[1][v];
            region = 3;
        } else {
            for (v = 0; v < 8; v++) F[v] = Fp[1][v] + S[1] * (Us[1][v] - U[1][v]);
            region = 4;
        }
        F[4] = 0.0;   /* the normal-field component carries no flux */
        if (uct) {   /* R19 */
            double chi[2], nu[2], nus, den, al, ar;
            for (a = 0; a < 2; a++) {
                chi[a] = (Va[a][1] - SM) * (S[a] - SM) / (Sa[a] + S[a] - 2.0 * SM);
                nu[a]  = (Sa[a] + S[a]) / (fabs(Sa[a]) + fabs(S[a]));
            }
            den = fabs(Sa[1]) + fabs(Sa[0]);
            nus = den > 0.0 ? (Sa[1] + Sa[0]) / den : 0.0;
            al = 0.5 * (1.0 + nus); ar = 0.5 * (1.0 - nus);
            uct[0] = al;
            uct[1] = 0.5 * (nu[0] - nus) * chi[0] + 0.5 * (fabs(Sa[0]) - nus * Sa[0]);
            uct[2] = 0.5 * (nu[1] - nus) * chi[1] + 0.5 * (fabs(Sa[1]) - nus * Sa[1]);
            uct[3] = al * VL[2] + ar * VR[2];
            uct[4] = al * VL[3] + ar * VR[3];
        }
        if (dbg) {
            dbg[2] = SM; dbg[3] = pTs; dbg[4] = Sa[0]; dbg[5] = Sa[1];
            for (v = 0; v < 8; v++) {
                dbg[24 + v] = Us[0][v]; dbg[32 + v] = Us[1][v];
                dbg[40 + v] = Uss[0][v]; dbg[48 + v] = Uss[1][v];
            }
        }
    }
    if (dbg) dbg[6] = (double)region;

    /* continuous upwind weight (R6) */
    wgt = 0.5 + 0.5 * F[0] / (THETA * fref);
    if (wgt < 0.0) wgt = 0.0;
    if (wgt > 1.0) wgt = 1.0;
    if (wout) *wout = wgt;
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ context */

static void free_all(void)
{
    int d;
    free(g.U); free(g.U1); free(g.U2);
    for (d = 0; d < 3; d++) { free(g.b[d]); free(g.b1[d]); free(g.b2[d]); }
    free(g.V); free(g.F); free(g.W); free(g.Eg); free(g.Ec); free(g.Uct);
    free(g.psi); free(g.psi1); free(g.psi2); free(g.Fpsi);
    memset(&g, 0, sizeof g);
}

static void set_dx(void)
{
    int d;
    for (d = 0; d < 3; d++) g.dx[d] = g.L[d] / g.n[d];
}

int oracle_init(int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter)
{
    int d, thr = g.threads;
    size_t N;
    if (g.init) free_all();
    g.threads = thr;
    if (nx < 1 || ny < 1 || nz < 1 || ghost < 2) return ORACLE_EINVAL;
    if (!(gamma > 1.0) || !(cfl > 0.0) || (limiter < 0 || limiter > 2)) return ORACLE_EINVAL;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    for (d = 0; d < 3; d++) g.act[d] = g.n[d] > 1;
    /* default box (R11): Lx = 1 and cubic cells */
    for (d = 0; d < 3; d++) g.L[d] = (double)g.n[d] / (double)nx;
    set_dx();
    g.gamma = gamma; g.cfl = cfl; g.limiter = limiter;
    N = (size_t)nx * ny * nz;
    g.N = N;
    g.U  = calloc(8 * N, sizeof(double));
    g.U1 = calloc(8 * N, sizeof(double));
    g.U2 = calloc(8 * N, sizeof(double));
    for (d = 0; d < 3; d++) {
        g.b[d]  = calloc(N, sizeof(double));
        g.b1[d] = calloc(N, sizeof(double));
        g.b2[d] = calloc(N, sizeof(double));
    }
    g.V  = calloc(8 * N, sizeof(double));
    g.F  = calloc(24 * N, sizeof(double));
    g.W  = calloc(3 * N, sizeof(double));
    g.Eg = calloc(3 * N, sizeof(double));
    g.Ec = calloc(3 * N, sizeof(double));
    g.Uct = calloc(15 * N, sizeof(double));
    g.psi = calloc(N, sizeof(double)); g.psi1 = calloc(N, sizeof(double)); g.psi2 = calloc(N, sizeof(double));
    g.Fpsi = calloc(3 * N, sizeof(double));
    if (!g.U || !g.U1 || !g.U2 || !g.V || !g.F || !g.W || !g.Eg || !g.Ec || !g.Uct) { free_all(); return ORACLE_ENOMEM; }
    if (!g.psi || !g.psi1 || !g.psi2 || !g.Fpsi) { free_all(); return ORACLE_ENOMEM; }
    for (d = 0; d < 3; d++) if (!g.b[d] || !g.b1[d] || !g.b2[d]) { free_all(); return ORACLE_ENOMEM; }
    g.init = 1;
    g.time = 0.0; g.dt_last = 0.0; g.stepped = 0; g.err = 0;
    return ORACLE_OK;
}

int oracle_finalize(void) { int t = g.threads; free_all(); g.threads = t; return ORACLE_OK; }

int oracle_set_threads(int n)
{
    g.threads = n > 0 ? n : 0;
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#endif
    return ORACLE_OK;
}

int oracle_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int oracle_set_box(double Lx, double Ly, double Lz)
{
    if (!g.init) return ORACLE_ESTATE;
    if (!(Lx > 0.0) || !(Ly > 0.0) || !(Lz > 0.0)) return ORACLE_EINVAL;
    g.L[0] = Lx; g.L[1] = Ly; g.L[2] = Lz;
    set_dx();
    return ORACLE_OK;
}

/* cell-centred B of each active direction := mean of its two faces (R7) */
static void cell_b_from_faces(double *U, double *const b[3])
{
    int d;
    for (d = 0; d < 3; d++) {
        long c;
        if (!g.act[d]) continue;
#pragma omp parallel for
        for (c = 0; c < (long)g.N; c++) {
            int i, j, k;
            c2ijk((size_t)c, &i, &j, &k);
            U[(4 + d) * g.N + c] = 0.5 * (b[d][c] + b[d][shift(i, j, k, d, +1)]);
        }
    }
}

static size_t face_count(int d)
{
    size_t m = 1; int e;
    for (e = 0; e < 3; e++) m *= (size_t)(g.n[e] + (e == d ? 1 : 0));
    return m;
}

int oracle_set_state(const double *U, const double *Bface)
{
    int d;
    size_t off = 0;
    if (!g.init) return ORACLE_ESTATE;
    if (!U) return ORACLE_EINVAL;
    memcpy(g.U, U, 8 * g.N * sizeof(double));
    if (g.divb == 1) {       /* GLM: the cell-centred B of U is the field; no faces; psi starts at zero */
        memset(g.psi, 0, g.N * sizeof(double));
        g.time = 0.0; g.stepped = 0; g.err = 0; g.dt_last = 0.0;
        return ORACLE_OK;
    }
    for (d = 0; d < 3; d++) {
        int i, j, k, m[3];
        if (!g.act[d]) continue;
        if (!Bface) return ORACLE_EINVAL;
        m[0] = g.n[0]; m[1] = g.n[1]; m[2] = g.n[2]; m[d] += 1;
        for (k = 0; k < g.n[2]; k++)
            for (j = 0; j < g.n[1]; j++)
                for (i = 0; i < g.n[0]; i++)
                    g.b[d][cidx(i, j, k)] = Bface[off + ((size_t)k * m[1] + j) * m[0] + i];
        off += face_count(d);
    }
    cell_b_from_faces(g.U, g.b);
    g.time = 0.0; g.stepped = 0; g.err = 0; g.dt_last = 0.0;
    return ORACLE_OK;
}

int oracle_get_state(double *U, double *Bface)
{
    int d;
    size_t off = 0;
    if (!g.init) return ORACLE_ESTATE;
    if (U) memcpy(U, g.U, 8 * g.N * sizeof(double));
    for (d = 0; d < 3; d++) {
        int i, j, k, m[3];
        if (!g.act[d]) continue;
        if (!Bface || g.divb == 1) break;
        m[0] = g.n[0]; m[1] = g.n[1]; m[2] = g.n[2]; m[d] += 1;
        for (k = 0; k < m[2]; k++)
            for (j = 0; j < m[1]; j++)
                for (i = 0; i < m[0]; i++)
                    Bface[off + ((size_t)k * m[1] + j) * m[0] + i] = g.b[d][cidx(i, j, k)];
        off += face_count(d);
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------ the scheme */

/* primitives of every cell (Eq. 7); returns nonzero if any cell is unphysical */
static int all_prims(const double *U, double *V)
{
    long c; int bad = 0;
#pragma omp parallel for reduction(|:bad)
    for (c = 0; c < (long)g.N; c++) {
        double u[8], q[8]; int v;
        for (v = 0; v < 8; v++) u[v] = U[v * g.N + c];
        if (oracle_cons2prim(u, g.gamma, q) != ORACLE_OK) bad |= 1;
        for (v = 0; v < 8; v++) V[v * g.N + c] = q[v];
    }
    return bad;
}

/* R8: dt = cfl / max_{cells, active d} ( (|v_d| + c_f,d) * (1/dx_d) ) */
static double cfl_dt(const double *U)
{
    long c; int d;
    double idx[3], smax = 0.0;
    if (all_prims(U, g.V)) g.err = 1;
    for (d = 0; d < 3; d++) idx[d] = 1.0 / g.dx[d];
#pragma omp parallel for reduction(max:smax)
    for (c = 0; c < (long)g.N; c++) {
        int dd;
        const double *V = g.V; size_t N = g.N;
        for (dd = 0; dd < 3; dd++) {
            int t1 = (dd + 1) % 3, t2 = (dd + 2) % 3;
            double cf, s;
            if (!g.act[dd]) continue;
            cf = oracle_fast_speed(V[c], V[7 * N + c], V[(4 + dd) * N + c], V[(4 + t1) * N + c], V[(4 + t2) * N + c], g.gamma);
            s = (fabs(V[(1 + dd) * N + c]) + cf) * idx[dd];
            if (s > smax) smax = s;
        }
    }
    return g.cfl / smax;
}

/* values at the edge between positions m1 and p0 of a quantity Q on a line of positions (m3, m2, m1 | p0, p1, p2):
   from below (the upper-face value of m1) and from above (the lower-face value of p0), with the reconstruction
   of the run: PLM (R4) or WENO-Z (R18) */
static void edge_values(const double *Q, size_t m3, size_t m2, size_t m1, size_t p0, size_t p1, size_t p2,
                        double *below, double *above)
{
    if (g.limiter == 2) {
        double sl[5] = { Q[m3], Q[m2], Q[m1], Q[p0], Q[p1] };
        double sr[5] = { Q[p2], Q[p1], Q[p0], Q[m1], Q[m2] };
        *below = oracle_wenoz(sl);
        *above = oracle_wenoz(sr);
    } else {
        *below = Q[m1] + 0.5 * oracle_plm_slope(Q[m1] - Q[m2], Q[p0] - Q[m1], g.limiter);
        *above = Q[p0] - 0.5 * oracle_plm_slope(Q[p0] - Q[m1], Q[p1] - Q[p0], g.limiter);
    }
}

/* UCT-HLLD edge EMF (reading R19; [47] named at PAPER.md:271, reference entry :640).  Component e at the edge
   (a-1/2, b-1/2) of cell c, (e,a,b) cyclic, E_e = v_b B_a - v_a B_b.  In the notation of the general upwind
   constrained-transport composition (W/E = below/above the edge along a, S/N = below/above it along b):

       E_e = -[ a_a^W (vbar_a B_b)^W + a_a^E (vbar_a B_b)^E ] + [ a_b^S (vbar_b B_a)^S + a_b^N (vbar_b B_a)^N ]
             + (d_a^E B_b^E - d_a^W B_b^W) - (d_b^N B_a^N - d_b^S B_a^S)

   - B_b^{W,E}: the staggered field b_b on the two b-faces that meet at the edge, reconstructed along a up to the
     edge from below (W) and from above (E); vbar_a^{W,E}: the transverse velocity a^L v_a^L + a^R v_a^R of the
     Riemann problems on those same b-faces, reconstructed the same way.  Likewise B_a, vbar_b on the two a-faces
     along b.  Reconstruction: the operator of the run (PLM with its limiter, or WENO-Z), as for the cell
     states -- with any other operator a grid-aligned run would not reproduce the 1D solution.
   - a_a^{W,E}, d_a^{W,E}: the coefficients a^L, a^R, d^L, d^R of the two a-interfaces that meet at the edge,
     arithmetic mean of the two; likewise for b.
   For data that does not vary along b this is the 1D formula of oracle_hlld_uct, i.e. -F_a[B_b] of HLLD. */
static void uct_edge_emf(int e, double *const bin[3])
{
    const size_t N = g.N;
    const int a = (e + 1) % 3, b = (e + 2) % 3;
    /* face data of direction d: [d][0] a^L, [1] d^L, [2] d^R, [3] vbar_t1, [4] vbar_t2 with (t1,t2) = (d+1,d+2):
       on a-faces vbar_b is t1 of a; on b-faces vbar_a is t2 of b */
    const double *aLa = g.Uct + ((size_t)a * 5 + 0) * N, *dLa = g.Uct + ((size_t)a * 5 + 1) * N, *dRa = g.Uct + ((size_t)a * 5 + 2) * N;
    const double *aLb = g.Uct + ((size_t)b * 5 + 0) * N, *dLb = g.Uct + ((size_t)b * 5 + 1) * N, *dRb = g.Uct + ((size_t)b * 5 + 2) * N;
    const double *vb_on_a = g.Uct + ((size_t)a * 5 + 3) * N;
    const double *va_on_b = g.Uct + ((size_t)b * 5 + 4) * N;
    const double *Ba = bin[a], *Bb = bin[b];
    double *Ee = g.Eg + (size_t)e * N;
    long c;
#pragma omp parallel for
    for (c = 0; c < (long)N; c++) {
        int i, j, k;
        size_t c11, c01, c10, am2, ap1, bm2, bp1, am3, ap2, bm3, bp2;
        double aW, aE, dW, dE, aS, aN, dS, dN;
        double BbW, BbE, vaW, vaE, BaS, BaN, vbS, vbN;
        c2ijk((size_t)c, &i, &j, &k);
        c11 = (size_t)c;
        c01 = shift(i, j, k, a, -1); am2 = shift(i, j, k, a, -2); ap1 = shift(i, j, k, a, +1);
        c10 = shift(i, j, k, b, -1); bm2 = shift(i, j, k, b, -2); bp1 = shift(i, j, k, b, +1);
        am3 = shift(i, j, k, a, -3); ap2 = shift(i, j, k, a, +2);
        bm3 = shift(i, j, k, b, -3); bp2 = shift(i, j, k, b, +2);
        /* a-interfaces below (c10) and above (c11) the edge along b; b-interfaces below (c01) / above (c11) along a */
        aW = 0.5 * (aLa[c10] + aLa[c11]); aE = 0.5 * ((1.0 - aLa[c10]) + (1.0 - aLa[c11]));
        dW = 0.5 * (dLa[c10] + dLa[c11]); dE = 0.5 * (dRa[c10] + dRa[c11]);
        aS = 0.5 * (aLb[c01] + aLb[c11]); aN = 0.5 * ((1.0 - aLb[c01]) + (1.0 - aLb[c11]));
        dS = 0.5 * (dLb[c01] + dLb[c11]); dN = 0.5 * (dRb[c01] + dRb[c11]);
        /* b-face quantities along a (cells am3, am2, c01 | edge | c11, ap1, ap2), a-face quantities along b */
        edge_values(Bb, am3, am2, c01, c11, ap1, ap2, &BbW, &BbE);
        edge_values(va_on_b, am3, am2, c01, c11, ap1, ap2, &vaW, &vaE);
        edge_values(Ba, bm3, bm2, c10, c11, bp1, bp2, &BaS, &BaN);
        edge_values(vb_on_a, bm3, bm2, c10, c11, bp1, bp2, &vbS, &vbN);
        Ee[c] = -(aW * vaW * BbW + aE * vaE * BbE) + (aS * vbS * BaS + aN * vbN * BaN)
                + (dE * BbE - dW * BbW) - (dN * BaN - dS * BaS);
    }
}

/* Euler(S, dt): (Uin, bin) -> (Uout, bout); fills g.V, g.F, g.W, g.Eg, g.Ec */
static void euler(const double *Uin, double *const bin[3], double dt, double *Uout, double *const bout[3])
{
    const size_t N = g.N;
    int d, e;
    long c;

    /* 1. primitives */
    if (all_prims(Uin, g.V)) g.err = 1;
    memset(g.F, 0, 24 * N * sizeof(double));
    memset(g.W, 0, 3 * N * sizeof(double));
    memset(g.Eg, 0, 3 * N * sizeof(double));

    /* 2. reconstruct + Riemann, direction by direction (Eq. 6, Eq. 8) */
    for (d = 0; d < 3; d++) {
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        /* the 7 reconstructed primitives in rotated order: rho, u, v, w, Bt1, Bt2, p */
        const int qv[7] = { 0, 1 + d, 1 + t1, 1 + t2, 4 + t1, 4 + t2, 7 };
        double *Fd = g.F + (size_t)d * 8 * N;
        double *Wd = g.W + (size_t)d * N;
        if (!g.act[d]) continue;
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k, q;
            size_t cm3, cm2, cm1, c0, cp1, cp2;
            double VL[7], VR[7], Fr[8], w;
            c2ijk((size_t)c, &i, &j, &k);
            cm2 = shift(i, j, k, d, -2); cm1 = shift(i, j, k, d, -1);
            c0 = (size_t)c;              cp1 = shift(i, j, k, d, +1);
            cm3 = shift(i, j, k, d, -3); cp2 = shift(i, j, k, d, +2);
            for (q = 0; q < 7; q++) {
                const double *Q = g.V + (size_t)qv[q] * N;
                if (g.limiter == 2) {          /* WENOZ (R18): q^L from the stencil of cell c-1, q^R from cell c mirrored */
                    double sl[5] = { Q[cm3], Q[cm2], Q[cm1], Q[c0], Q[cp1] };
                    double sr[5] = { Q[cp2], Q[cp1], Q[c0], Q[cm1], Q[cm2] };
                    VL[q] = oracle_wenoz(sl);
                    VR[q] = oracle_wenoz(sr);
                    continue;
                }
                /* slope of cell c-1 and of cell c (R4) */
                double sm = oracle_plm_slope(Q[cm1] - Q[cm2], Q[c0] - Q[cm1], g.limiter);
                double s0 = oracle_plm_slope(Q[c0] - Q[cm1], Q[cp1] - Q[c0], g.limiter);
                VL[q] = Q[cm1] + 0.5 * sm;     /* q^L at (c-1)+1/2, Eq. 6 */
                VR[q] = Q[c0] - 0.5 * s0;      /* q^R at c-1/2 */
            }
            /* interface c-1/2: normal field is the face value on both sides (R7) */
            if (g.emf == 1) {
                double uct[5]; int m;
                oracle_hlld_uct(VL, VR, bin[d][c0], g.gamma, Fr, &w, NULL, uct);
                for (m = 0; m < 5; m++) g.Uct[((size_t)d * 5 + m) * N + c0] = uct[m];
            } else
            oracle_hlld(VL, VR, bin[d][c0], g.gamma, Fr, &w, NULL);
            /* rotate back to lab components */
            Fd[0 * N + c0] = Fr[0];
            Fd[(1 + d) * N + c0] = Fr[1]; Fd[(1 + t1) * N + c0] = Fr[2]; Fd[(1 + t2) * N + c0] = Fr[3];
            Fd[(4 + d) * N + c0] = 0.0;   Fd[(4 + t1) * N + c0] = Fr[5]; Fd[(4 + t2) * N + c0] = Fr[6];
            Fd[7 * N + c0] = Fr[7];
            Wd[c0] = w;
        }
    }

    /* 3. flux-difference update, x then y then z (Eq. 4, Fig. 2) */
    memcpy(Uout, Uin, 8 * N * sizeof(double));
    for (d = 0; d < 3; d++) {
        const double *Fd = g.F + (size_t)d * 8 * N;
        double dtdx;
        if (!g.act[d]) continue;
        dtdx = dt / g.dx[d];
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k, v; size_t cp1;
            c2ijk((size_t)c, &i, &j, &k);
            cp1 = shift(i, j, k, d, +1);
            for (v = 0; v < 8; v++)
                Uout[v * N + c] -= dtdx * (Fd[v * N + cp1] - Fd[v * N + c]);
        }
    }

    /* 4. constrained transport (R6) */
    /* cell-centred EMF  E^c = -v x B */
#pragma omp parallel for
    for (c = 0; c < (long)N; c++) {
        const double *V = g.V;
        double vx = V[1 * N + c], vy = V[2 * N + c], vz = V[3 * N + c];
        double Bx = V[4 * N + c], By = V[5 * N + c], Bz = V[6 * N + c];
        g.Ec[0 * N + c] = vz * By - vy * Bz;
        g.Ec[1 * N + c] = vx * Bz - vz * Bx;
        g.Ec[2 * N + c] = vy * Bx - vx * By;
    }
    /* edge EMF component e lives at (a-1/2, b-1/2) of cell c, (e,a,b) cyclic */
    for (e = 0; e < 3; e++) {
        const int a = (e + 1) % 3, b = (e + 2) % 3;
        const double *Fa = g.F + (size_t)a * 8 * N + (size_t)(4 + b) * N;   /* F_a[B_b] */
        const double *Fb = g.F + (size_t)b * 8 * N + (size_t)(4 + a) * N;   /* F_b[B_a] */
        const double *Wa = g.W + (size_t)a * N, *Wb = g.W + (size_t)b * N;
        const double *Ec = g.Ec + (size_t)e * N;
        double *Ee = g.Eg + (size_t)e * N;
        if (!(g.act[a] && g.act[b])) continue;
        if (g.emf == 1) { uct_edge_emf(e, bin); continue; }
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k, q[3];
            size_t c11, c01, c10, c00;
            double Ea_lo, Ea_hi, Eb_lo, Eb_hi, wa_lo, wa_hi, wb_lo, wb_hi;
            double t1, t2, t3, t4;
            c2ijk((size_t)c, &i, &j, &k);
            c11 = (size_t)c;                         /* cell (ia  , ib  ) */
            c01 = shift(i, j, k, a, -1);             /* cell (ia-1, ib  ) */
            c10 = shift(i, j, k, b, -1);             /* cell (ia  , ib-1) */
            q[0] = i; q[1] = j; q[2] = k; q[a] -= 1; q[b] -= 1;
            c00 = cidx(q[0], q[1], q[2]);            /* cell (ia-1, ib-1) */
            /* face EMFs: on a-faces E_e = -F_a[B_b], on b-faces E_e = +F_b[B_a] */
            Ea_lo = -Fa[c10]; Ea_hi = -Fa[c11];
            Eb_lo =  Fb[c01]; Eb_hi =  Fb[c11];
            wa_lo = Wa[c10]; wa_hi = Wa[c11];
            wb_lo = Wb[c01]; wb_hi = Wb[c11];
            /* up(w; lower-cell value, upper-cell value) = w*lower + (1-w)*upper */
            t1 = wa_lo * (Eb_lo - Ec[c00]) + (1.0 - wa_lo) * (Eb_hi - Ec[c10]);
            t2 = wa_hi * (Ec[c01] - Eb_lo) + (1.0 - wa_hi) * (Ec[c11] - Eb_hi);
            t3 = wb_lo * (Ea_lo - Ec[c00]) + (1.0 - wb_lo) * (Ea_hi - Ec[c01]);
            t4 = wb_hi * (Ec[c10] - Ea_lo) + (1.0 - wb_hi) * (Ec[c11] - Ea_hi);
            Ee[c] = 0.25 * (Ea_lo + Ea_hi + Eb_lo + Eb_hi) + 0.25 * (t1 - t2) + 0.25 * (t3 - t4);
        }
    }
    /* face update  db_d/dt = -(curl E)_d, terms of inactive dimensions dropped */
    for (d = 0; d < 3; d++) {
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        const double *E1 = g.Eg + (size_t)t1 * N, *E2 = g.Eg + (size_t)t2 * N;
        if (!g.act[d]) { continue; }
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k;
            double term1 = 0.0, term2 = 0.0;
            c2ijk((size_t)c, &i, &j, &k);
            if (g.act[t1]) term1 = (E2[shift(i, j, k, t1, +1)] - E2[c]) / g.dx[t1];
            if (g.act[t2]) term2 = (E1[shift(i, j, k, t2, +1)] - E1[c]) / g.dx[t2];
            bout[d][c] = bin[d][c] - dt * (term1 - term2);
        }
    }
    /* 5. cell-centred B of the active dimensions from the new faces; E untouched (R7) */
    cell_b_from_faces(Uout, bout);
}


/* ------------------------------------------------------------------ GLM divergence cleaning (R20)
 * The paper's other divergence control ("divergence cleaning [43, 44]", used in its strong-scaling
 * runs) is named, not printed.  Reading R20 restates the mixed hyperbolic / parabolic GLM-MHD
 * scheme of Dedner et al. 2002 [43] in its conservative form:
 *     dB/dt + div(v B - B v) + grad psi = 0,      dpsi/dt + c_h^2 div B = -(c_h^2 / c_p^2) psi,
 * cell-centred B, one extra scalar psi, no face fields, no CT.  Per interface, the (B_n, psi) pair obeys a
 * linear 2x2 system with the waves -c_h, +c_h whatever the fluid does; its Riemann problem is solved exactly,
 *     B_m   = (B_nL + B_nR)/2 - (psi_R - psi_L)/(2 c_h),      psi_m = (psi_L + psi_R)/2 - c_h (B_nR - B_nL)/2,
 * the flux of B_n is psi_m and the flux of psi is c_h^2 B_m, and the other seven fluxes are the HLLD fluxes
 * with the normal field B_m on both sides.  c_h = cfl * min_d(dx_d) / dt (the fastest speed the time step
 * allows); after every full step psi is damped exactly, psi *= exp(-dt c_h / c_r), with the constant
 * c_r = c_p^2 / c_h = 0.18 that [43] recommends.  The energy equation is unchanged (total energy conserved). */
#define GLM_CR 0.18

void oracle_glm_interface(double BnL, double BnR, double psiL, double psiR, double ch, double *Bm, double *psim)
{
    *Bm = 0.5 * (BnL + BnR) - 0.5 * (psiR - psiL) / ch;
    *psim = 0.5 * (psiL + psiR) - 0.5 * ch * (BnR - BnL);
}

static double glm_ch(double dt)
{
    int d; double h = 0.0;
    for (d = 0; d < 3; d++) if (g.act[d] && (h == 0.0 || g.dx[d] < h)) h = g.dx[d];
    return g.cfl * h / dt;
}

/* Euler(S, dt) of the GLM variant: (Uin, psin) -> (Uout, psout); fills g.V, g.F, g.Fpsi */
static void euler_glm(const double *Uin, const double *psin, double dt, double ch, double *Uout, double *psout)
{
    const size_t N = g.N;
    int d;
    long c;
    if (all_prims(Uin, g.V)) g.err = 1;
    memset(g.F, 0, 24 * N * sizeof(double));
    memset(g.Fpsi, 0, 3 * N * sizeof(double));
    for (d = 0; d < 3; d++) {
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        /* the 7 HLLD primitives in rotated order, then the normal field and psi */
        const int qv[8] = { 0, 1 + d, 1 + t1, 1 + t2, 4 + t1, 4 + t2, 7, 4 + d };
        double *Fd = g.F + (size_t)d * 8 * N;
        double *Fp = g.Fpsi + (size_t)d * N;
        if (!g.act[d]) continue;
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k, q;
            size_t cm3, cm2, cm1, c0, cp1, cp2;
            double VL[9], VR[9], Fr[8], w, Bm, psim;
            c2ijk((size_t)c, &i, &j, &k);
            cm2 = shift(i, j, k, d, -2); cm1 = shift(i, j, k, d, -1);
            c0 = (size_t)c;              cp1 = shift(i, j, k, d, +1);
            cm3 = shift(i, j, k, d, -3); cp2 = shift(i, j, k, d, +2);
            for (q = 0; q < 9; q++) {
                const double *Q = q < 8 ? g.V + (size_t)qv[q] * N : psin;
                if (g.limiter == 2) {
                    double sl[5] = { Q[cm3], Q[cm2], Q[cm1], Q[c0], Q[cp1] };
                    double sr[5] = { Q[cp2], Q[cp1], Q[c0], Q[cm1], Q[cm2] };
                    VL[q] = oracle_wenoz(sl);
                    VR[q] = oracle_wenoz(sr);
                } else {
                    double sm = oracle_plm_slope(Q[cm1] - Q[cm2], Q[c0] - Q[cm1], g.limiter);
                    double s0 = oracle_plm_slope(Q[c0] - Q[cm1], Q[cp1] - Q[c0], g.limiter);
                    VL[q] = Q[cm1] + 0.5 * sm;
                    VR[q] = Q[c0] - 0.5 * s0;
                }
            }
            /* interface c-1/2: exact (B_n, psi) state, then HLLD with that normal field on both sides */
            oracle_glm_interface(VL[7], VR[7], VL[8], VR[8], ch, &Bm, &psim);
            oracle_hlld(VL, VR, Bm, g.gamma, Fr, &w, NULL);
            Fd[0 * N + c0] = Fr[0];
            Fd[(1 + d) * N + c0] = Fr[1]; Fd[(1 + t1) * N + c0] = Fr[2]; Fd[(1 + t2) * N + c0] = Fr[3];
            Fd[(4 + d) * N + c0] = psim;  Fd[(4 + t1) * N + c0] = Fr[5]; Fd[(4 + t2) * N + c0] = Fr[6];
            Fd[7 * N + c0] = Fr[7];
            Fp[c0] = ch * ch * Bm;
        }
    }
    memcpy(Uout, Uin, 8 * N * sizeof(double));
    memcpy(psout, psin, N * sizeof(double));
    for (d = 0; d < 3; d++) {
        const double *Fd = g.F + (size_t)d * 8 * N;
        const double *Fp = g.Fpsi + (size_t)d * N;
        double dtdx;
        if (!g.act[d]) continue;
        dtdx = dt / g.dx[d];
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) {
            int i, j, k, v; size_t cp1;
            c2ijk((size_t)c, &i, &j, &k);
            cp1 = shift(i, j, k, d, +1);
            for (v = 0; v < 8; v++)
                Uout[v * N + c] -= dtdx * (Fd[v * N + cp1] - Fd[v * N + c]);
            psout[c] -= dtdx * (Fp[cp1] - Fp[c]);
        }
    }
}

static void one_step_glm(double dt)
{
    const size_t N = g.N;
    const double ch = glm_ch(dt);
    const double damp = exp(-dt * ch / GLM_CR);
    long c;
    if (g.rk_order == 3) {      /* Eq. 5 (R17), as in one_step */
        euler_glm(g.U, g.psi, dt, ch, g.U1, g.psi1);
        euler_glm(g.U1, g.psi1, dt, ch, g.U2, g.psi2);
#pragma omp parallel for
        for (c = 0; c < (long)(8 * N); c++) g.U2[c] = (3.0 * g.U[c] + g.U2[c]) / 4.0;
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) g.psi2[c] = (3.0 * g.psi[c] + g.psi2[c]) / 4.0;
        euler_glm(g.U2, g.psi2, dt, ch, g.U1, g.psi1);
#pragma omp parallel for
        for (c = 0; c < (long)(8 * N); c++) g.U[c] = (g.U[c] + 2.0 * g.U1[c]) / 3.0;
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) g.psi[c] = (g.psi[c] + 2.0 * g.psi1[c]) / 3.0;
    } else {                    /* R3 */
        euler_glm(g.U, g.psi, dt, ch, g.U1, g.psi1);
        euler_glm(g.U1, g.psi1, dt, ch, g.U2, g.psi2);
#pragma omp parallel for
        for (c = 0; c < (long)(8 * N); c++) g.U[c] = 0.5 * (g.U[c] + g.U2[c]);
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) g.psi[c] = 0.5 * (g.psi[c] + g.psi2[c]);
    }
    /* the parabolic part of the psi equation, integrated exactly over the step */
#pragma omp parallel for
    for (c = 0; c < (long)N; c++) g.psi[c] *= damp;
    g.time += dt;
    g.dt_last = dt;
    g.stepped = 1;
}

int oracle_set_emf(int mode)
{
    if (!g.init) return ORACLE_ESTATE;
    if (mode != 0 && mode != 1) return ORACLE_EINVAL;
    g.emf = mode;
    return ORACLE_OK;
}

int oracle_set_divb(int mode)
{
    if (!g.init) return ORACLE_ESTATE;
    if (mode != 0 && mode != 1) return ORACLE_EINVAL;
    g.divb = mode;
    return ORACLE_OK;
}

int oracle_set_psi(const double *psi)
{
    if (!g.init || g.divb != 1) return ORACLE_ESTATE;
    memcpy(g.psi, psi, g.N * sizeof(double));
    return ORACLE_OK;
}

int oracle_get_psi(double *psi)
{
    if (!g.init || g.divb != 1) return ORACLE_ESTATE;
    memcpy(psi, g.psi, g.N * sizeof(double));
    return ORACLE_OK;
}

static void one_step(double dt)
{
    const size_t N = g.N;
    long c; int d;
    if (g.divb == 1) { one_step_glm(dt); return; }
    if (g.rk_order == 3) {
        /* Eq. 5, SSP-RK3 in Shu-Osher form; reading R17: the last stage carries 2 L**
           (as printed, "+ L**", the weights of L do not sum to one):
             U*  = U^n + L^n ;  U** = (3 U^n + U* + L*) / 4 ;  U^{n+1} = (U^n + 2 (U** + L**)) / 3 */
        euler(g.U, g.b, dt, g.U1, g.b1);                 /* U1 = U*            */
        euler(g.U1, g.b1, dt, g.U2, g.b2);               /* U2 = U* + L*       */
#pragma omp parallel for
        for (c = 0; c < (long)(8 * N); c++) g.U2[c] = (3.0 * g.U[c] + g.U2[c]) / 4.0;
        for (d = 0; d < 3; d++) {
            if (!g.act[d]) continue;
#pragma omp parallel for
            for (c = 0; c < (long)N; c++) g.b2[d][c] = (3.0 * g.b[d][c] + g.b2[d][c]) / 4.0;
        }
        cell_b_from_faces(g.U2, g.b2);                   /* U2 = U**           */
        euler(g.U2, g.b2, dt, g.U1, g.b1);               /* U1 = U** + L**     */
#pragma omp parallel for
        for (c = 0; c < (long)(8 * N); c++) g.U[c] = (g.U[c] + 2.0 * g.U1[c]) / 3.0;
        for (d = 0; d < 3; d++) {
            if (!g.act[d]) continue;
#pragma omp parallel for
            for (c = 0; c < (long)N; c++) g.b[d][c] = (g.b[d][c] + 2.0 * g.b1[d][c]) / 3.0;
        }
        cell_b_from_faces(g.U, g.b);
        g.time += dt;
        g.dt_last = dt;
        g.stepped = 1;
        return;
    }
    /* R3: U* = U^n + L^n ; U^{n+1} = (U^n + U* + L*) / 2, same dt in both stages */
    euler(g.U, g.b, dt, g.U1, g.b1);
    euler(g.U1, g.b1, dt, g.U2, g.b2);
#pragma omp parallel for
    for (c = 0; c < (long)(8 * N); c++) g.U[c] = 0.5 * (g.U[c] + g.U2[c]);
    for (d = 0; d < 3; d++) {
        if (!g.act[d]) continue;
#pragma omp parallel for
        for (c = 0; c < (long)N; c++) g.b[d][c] = 0.5 * (g.b[d][c] + g.b2[d][c]);
    }
    cell_b_from_faces(g.U, g.b);
    g.time += dt;
    g.dt_last = dt;
    g.stepped = 1;
}

/* time integrator: 2 = SSP-RK2 (north_star, default), 3 = SSP-RK3 of Eq. 5 */
int oracle_set_integrator(int order)
{
    if (order != 2 && order != 3) return ORACLE_EINVAL;
    g.rk_order = order;
    return ORACLE_OK;
}

int oracle_step(int nsteps)
{
    int s;
    if (!g.init) return ORACLE_ESTATE;
    if (nsteps < 0) return ORACLE_EINVAL;
    for (s = 0; s < nsteps; s++) {
        double dt = cfl_dt(g.U);
        one_step(dt);
        if (g.err) return ORACLE_EPHYS;
    }
    return g.err ? ORACLE_EPHYS : ORACLE_OK;
}

int oracle_step_fixed_dt(int nsteps, double dt)
{
    int s;
    if (!g.init) return ORACLE_ESTATE;
    if (nsteps < 0 || !(dt > 0.0)) return ORACLE_EINVAL;
    for (s = 0; s < nsteps; s++) {
        one_step(dt);
        if (g.err) return ORACLE_EPHYS;
    }
    return ORACLE_OK;
}

double oracle_get_dt(void)
{
    if (!g.init) return NAN;
    if (g.stepped) return g.dt_last;
    return cfl_dt(g.U);
}

double oracle_get_time(void) { return g.init ? g.time : NAN; }

int oracle_debug_euler(double dt, double *U1, double *Bf1, double *F, double *W, double *Eedge)
{
    const size_t N = g.N;
    int d;
    if (!g.init) return ORACLE_ESTATE;
    euler(g.U, g.b, dt, g.U1, g.b1);
    if (U1) memcpy(U1, g.U1, 8 * N * sizeof(double));
    if (Bf1) {
        size_t off = 0;
        for (d = 0; d < 3; d++) {
            int i, j, k, m[3];
            if (!g.act[d]) continue;
            m[0] = g.n[0]; m[1] = g.n[1]; m[2] = g.n[2]; m[d] += 1;
            for (k = 0; k < m[2]; k++)
                for (j = 0; j < m[1]; j++)
                    for (i = 0; i < m[0]; i++)
                        Bf1[off + ((size_t)k * m[1] + j) * m[0] + i] = g.b1[d][cidx(i, j, k)];
            off += face_count(d);
        }
    }
    if (F) memcpy(F, g.F, 24 * N * sizeof(double));
    if (W) memcpy(W, g.W, 3 * N * sizeof(double));
    if (Eedge) memcpy(Eedge, g.Eg, 3 * N * sizeof(double));
    return g.err ? ORACLE_EPHYS : ORACLE_OK;
}
