// glm.cuh -- the GLM divergence-cleaning variant of the step ("divergence
// cleaning [43, 44]", the divergence control of the paper's strong-scaling runs).
//
// Reading R20: the conservative mixed hyperbolic / parabolic GLM-MHD scheme of Dedner et al. 2002
// ([43]), restated from the published algorithm:
//     dB/dt + div(v B - B v) + grad psi = 0,      dpsi/dt + c_h^2 div B = -(c_h^2 / c_p^2) psi,
// cell-centred B (the three magnetic arrays of a state hold cell values), one more scalar psi, no face
// fields and no CT kernel.  At an interface the (B_n, psi) pair obeys a linear system with the waves -c_h and
// +c_h; its Riemann problem is solved exactly,
//     B_m = (B_nL + B_nR)/2 - (psi_R - psi_L)/(2 c_h),     psi_m = (psi_L + psi_R)/2 - c_h (B_nR - B_nL)/2,
// flux(B_n) = psi_m, flux(psi) = c_h^2 B_m, and the other seven fluxes are HLLD's with the normal field B_m.
// c_h = cfl min_d(dx_d) / dt; after a full step psi *= exp(-dt c_h / c_r), c_r = 0.18 ([43]'s recommendation).
//
// One launch per direction (not fused like the CT path): along x a block works on a row segment in shared memory
// (k_glm_sweep_x), along y and z a thread marches up its column (k_glm_march); every interface is solved once.  The
// last sweep of a combine stage applies the Runge-Kutta combine (a7) and the damping of psi itself and, at the end
// of a step, leaves the dt bound grid.
#pragma once
#include "kernels.cuh"

namespace pluto {

// kGlmCr (c_p^2 / c_h of [43]) lives in grid.h: k_dtfinish (dt_kernel.cu) forms the damping factor from it

// the nine stored values of one zone: rho, m_x, m_y, m_z, E, B_x, B_y, B_z, psi
__device__ __forceinline__ void glm_load(const Grid &g, const double *__restrict__ S, const double *__restrict__ psi,
                                         long long c, double u[9])
{
#pragma unroll
    for (int v = 0; v < 8; v++) u[v] = S[v * g.sa + c];
    u[8] = psi[c];
}

// rotated primitives of one zone for a sweep along DIR: rho, u, v, w, B_t1, B_t2, p, B_n, psi
template <int DIR>
__device__ __forceinline__ void glm_convert(const Grid &g, const double u[9], double q[9], bool &bad)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const double rho = u[0], En = u[4];
    const double m[3] = { u[1], u[2], u[3] };
    const double B[3] = { u[5], u[6], u[7] };
    const double ir = rcp_fast(rho);
    const double v[3] = { __dmul_rn(m[0], ir), __dmul_rn(m[1], ir), __dmul_rn(m[2], ir) };
    const double p = __dmul_rn(g.gamma - 1.0, fma(-0.5, fma(B[0], B[0], fma(B[1], B[1], B[2] * B[2])),
                                                  fma(-0.5, fma(m[0], v[0], fma(m[1], v[1], m[2] * v[2])), En)));
    q[0] = rho; q[1] = v[DIR]; q[2] = v[T1]; q[3] = v[T2]; q[4] = B[T1]; q[5] = B[T2]; q[6] = p; q[7] = B[DIR];
    q[8] = u[8];
    bad = unphysical(rho) || unphysical(p);
}

template <int DIR>
__device__ __forceinline__ void glm_prims(const Grid &g, const double *__restrict__ S, const double *__restrict__ psi,
                                          long long c, double q[9], bool &bad)
{
    double u[9];
    glm_load(g, S, psi, c, u);
    glm_convert<DIR>(g, u, q, bad);
}

// flux of the nine variables through one interface from the reconstructed states (rotated frame):
// f[0..6] = HLLD (rho, m_n, m_t1, m_t2, B_t1, B_t2, E), f[7] = flux of B_n, f[8] = flux of psi
__device__ __forceinline__ void glm_face_flux(const double L[9], const double R[9], double ch, double gamma, double igm1,
                                              double f[9])
{
    const double Bm = fma(-0.5, (R[8] - L[8]) * rcp_fast(ch), 0.5 * (L[7] + R[7]));
    const double psim = fma(-0.5 * ch, R[7] - L[7], 0.5 * (L[8] + R[8]));
    const Side sl = { L[0], L[1], L[2], L[3], L[4], L[5], L[6] };
    const Side sr = { R[0], R[1], R[2], R[3], R[4], R[5], R[6] };
    double w;
    hlld(sl, sr, Bm, gamma, igm1, f, w);
    f[7] = psim;
    f[8] = __dmul_rn(ch * ch, Bm);
}

// One direction of one Euler stage: out = (FIRST ? in : out) - dt/dx_DIR (F(+) - F(-)) for the nine variables.

// The x direction: a block takes GLMX_NT consecutive zones of one row (blocks overlap by four zones), every
// thread converts its zone once, limits its own slopes from its two neighbours' primitives in shared memory,
// solves the interface on its lower face with its left neighbour's upper-face value, and differences its flux
// with its right neighbour's: every interface once, three block barriers.
constexpr int GLMX_NT = 128;

template <int LIM, bool FIRST>
__global__ void __launch_bounds__(GLMX_NT, 4)
k_glm_sweep_x(Grid g, const double *__restrict__ Sin, const double *__restrict__ psin, double *Sout, double *psout,
              StepParams *P)
{
    __shared__ double sq[9][GLMX_NT];      // primitives, then the fluxes
    __shared__ double sh[9][GLMX_NT];      // upper-face values
    const int t = threadIdx.x, nx = g.n[0];
    const int i = (int)blockIdx.x * (GLMX_NT - 4) - 2 + t, j = blockIdx.y, k = blockIdx.z;
    const bool valid = i < nx + 2;
    const long long sa = g.sa, c = g.at(valid ? i : 0, j, k);
    const double ch = P->glm_ch, dtdx = P->dtdx[0];
    double u[9], q[9];
    bool bad;
    glm_load(g, Sin, psin, c, u);
    glm_convert<0>(g, u, q, bad);
    if (valid && i >= 0 && i < nx && bad) P->err = 1;
#pragma unroll
    for (int v = 0; v < 9; v++) sq[v][t] = q[v];
    __syncthreads();
    const bool has_nb = valid && t >= 1 && t <= GLMX_NT - 2 && i + 1 < nx + 2;
    double R[9];
    if (has_nb) {
#pragma unroll
        for (int v = 0; v < 9; v++) {
            double hi;
            plm_faces<LIM>(q[v], q[v] - sq[v][t - 1], sq[v][t + 1] - q[v], R[v], hi);
            sh[v][t] = hi;
        }
    }
    __syncthreads();
    const bool face = has_nb && t >= 2 && i >= 0;
    double F[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
    if (face) {
        const double L[9] = { sh[0][t - 1], sh[1][t - 1], sh[2][t - 1], sh[3][t - 1], sh[4][t - 1],
                              sh[5][t - 1], sh[6][t - 1], sh[7][t - 1], sh[8][t - 1] };
        glm_face_flux(L, R, ch, g.gamma, g.igm1, F);
#pragma unroll
        for (int v = 0; v < 9; v++) sq[v][t] = F[v];
    }
    __syncthreads();
    if (face && i < nx && t <= GLMX_NT - 3) {
        // rotated flux along x: (rho, m_x, m_y, m_z, B_y, B_z, E, B_x, psi); base = the zone's own stored values
        double b[9];
#pragma unroll
        for (int v = 0; v < 9; v++) b[v] = u[v];
        if (!FIRST) glm_load(g, Sout, psout, c, b);
        Sout[c] = fma(-dtdx, sq[0][t + 1] - F[0], b[0]);
        Sout[sa + c] = fma(-dtdx, sq[1][t + 1] - F[1], b[1]);
        Sout[2 * sa + c] = fma(-dtdx, sq[2][t + 1] - F[2], b[2]);
        Sout[3 * sa + c] = fma(-dtdx, sq[3][t + 1] - F[3], b[3]);
        Sout[4 * sa + c] = fma(-dtdx, sq[6][t + 1] - F[6], b[4]);
        Sout[5 * sa + c] = fma(-dtdx, sq[7][t + 1] - F[7], b[5]);
        Sout[6 * sa + c] = fma(-dtdx, sq[4][t + 1] - F[4], b[6]);
        Sout[7 * sa + c] = fma(-dtdx, sq[5][t + 1] - F[5], b[7]);
        psout[c] = fma(-dtdx, sq[8][t + 1] - F[8], b[8]);
    }
}

// The same update along y or z (DIR = 1, 2) by marching: thread = one column, the running PLM state of the
// nine primitives in registers, every interface solved once per segment (+1 at the segment end), every zone
// loaded and converted once -- the scheme of k_sweep_march (kernels.cuh) for the cell-centred variant.
// DIR = 1: grid.y = segment, grid.z = k;  DIR = 2: grid.y = j, grid.z = segment.
// COMB: this is the last sweep of a combine stage: the zone's result wn * S^n + ws * (base - dt/dx dF) goes to
// the stage's output arrays Fout / fpsout (which may be S^n itself: each value is read before the same thread
// overwrites it), psi also takes the damping factor at the end of a step; no separate combine pass.  BOUND (z march
// of the last stage): the dt upper bound of the zones a thread finishes, as in k_sweep_march.
struct GlmCombine { double *Fout, *fpsout; const double *Sn, *psn; double wn, ws; int do_damp; };

template <int DIR, int LIM, bool FIRST, bool COMB, bool BOUND>
__global__ void __launch_bounds__(128, 2)
k_glm_march(Grid g, const double *__restrict__ Sin, const double *__restrict__ psin, double *Sout, double *psout,
            StepParams *P, int seglen, GlmCombine cbg, BoundGrid bg)
{
    __shared__ double sbnd[BOUND ? 3 : 1][128];
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n[0]) return;
    const int seg = DIR == 1 ? blockIdx.y : blockIdx.z;
    const int tr = DIR == 1 ? blockIdx.z : blockIdx.y;
    const int s0 = seg * seglen, s1 = min(s0 + seglen, g.n[DIR]);
    const long long sa = g.sa, st = g.st[DIR];
    long long c = DIR == 1 ? g.at(i, s0, tr) : g.at(i, tr, s0);
    const double ch = P->glm_ch, dtdx = P->dtdx[DIR];
    const double *base = FIRST ? Sin : Sout;
    const double *pbase = FIRST ? psin : psout;
    bool bad, anybad = false;
    SigmaBound sb;
    if (BOUND) sb.init(&sbnd[0][threadIdx.x], 128);
    const double damp = (COMB && cbg.do_damp) ? P->glm_damp : 1.0;
    double q0[9], d0[9], qL[9];
    {
        double qm[9];
        glm_prims<DIR>(g, Sin, psin, c - 2 * st, qm, bad);
        glm_prims<DIR>(g, Sin, psin, c - st, q0, bad);
#pragma unroll
        for (int v = 0; v < 9; v++) d0[v] = q0[v] - qm[v];
        glm_prims<DIR>(g, Sin, psin, c, qm, bad);
        anybad |= bad;
#pragma unroll
        for (int v = 0; v < 9; v++) {
            double d1 = qm[v] - q0[v], lo;
            plm_faces<LIM>(q0[v], d0[v], d1, lo, qL[v]);
            q0[v] = qm[v];
            d0[v] = d1;
        }
    }
    double Fp[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
    // software pipeline: the stored values of zone s+1 (and the update base of zone s-1) are loaded one
    // iteration before they are used, so the march does not stall on memory
    double un[9], ub[9], us[9];
    glm_load(g, Sin, psin, c + st, un);
    glm_load(g, base, pbase, c - st, ub);
    if (COMB) glm_load(g, cbg.Sn, cbg.psn, c - st, us);
    for (int s = s0; s <= s1; s++, c += st) {
        double q1[9], qR[9], F[9], uc[9], bc[9], sc[9];
#pragma unroll
        for (int v = 0; v < 9; v++) { uc[v] = un[v]; bc[v] = ub[v]; if (COMB) sc[v] = us[v]; }
        if (s < s1) {
            glm_load(g, Sin, psin, c + 2 * st, un);
            glm_load(g, base, pbase, c, ub);
            if (COMB) glm_load(g, cbg.Sn, cbg.psn, c, us);
        }
        glm_convert<DIR>(g, uc, q1, bad);
        if (s + 1 < s1) anybad |= bad;
        const double L9[9] = { qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6], qL[7], qL[8] };
#pragma unroll
        for (int v = 0; v < 9; v++) {
            double d1 = q1[v] - q0[v];
            plm_faces<LIM>(q0[v], d0[v], d1, qR[v], qL[v]);
            q0[v] = q1[v];
            d0[v] = d1;
        }
        glm_face_flux(L9, qR, ch, g.gamma, g.igm1, F);
        if (s > s0) {
            const long long cm = c - st;
            // stored order: rho, m_x, m_y, m_z, E, B_x, B_y, B_z, psi; rotated flux: (rho, m_n, m_t1, m_t2, B_t1, B_t2, E, B_n, psi)
            double r[9];
            r[0] = fma(-dtdx, F[0] - Fp[0], bc[0]);
            r[1 + DIR] = fma(-dtdx, F[1] - Fp[1], bc[1 + DIR]);
            r[1 + T1] = fma(-dtdx, F[2] - Fp[2], bc[1 + T1]);
            r[1 + T2] = fma(-dtdx, F[3] - Fp[3], bc[1 + T2]);
            r[4] = fma(-dtdx, F[6] - Fp[6], bc[4]);
            r[5 + DIR] = fma(-dtdx, F[7] - Fp[7], bc[5 + DIR]);
            r[5 + T1] = fma(-dtdx, F[4] - Fp[4], bc[5 + T1]);
            r[5 + T2] = fma(-dtdx, F[5] - Fp[5], bc[5 + T2]);
            r[8] = fma(-dtdx, F[8] - Fp[8], bc[8]);
            if (COMB) {
#pragma unroll
                for (int v = 0; v < 9; v++) r[v] = fma(cbg.wn, sc[v], cbg.ws * r[v]);
                if (cbg.do_damp) r[8] *= damp;
#pragma unroll
                for (int v = 0; v < 8; v++) cbg.Fout[v * sa + cm] = r[v];
                cbg.fpsout[cm] = r[8];
            } else {
#pragma unroll
                for (int v = 0; v < 8; v++) Sout[v * sa + cm] = r[v];
                psout[cm] = r[8];
            }
            if (BOUND) sb.add(g, r[0], r[1], r[2], r[3], r[4]);
        }
#pragma unroll
        for (int v = 0; v < 9; v++) Fp[v] = F[v];
    }
    if (anybad) P->err = 1;
    if (BOUND) bound_publish(bg, DIR == 1 ? s0 : tr, DIR == 1 ? tr : s0, sb.value(g, bg.cfac));
}

} // namespace pluto
