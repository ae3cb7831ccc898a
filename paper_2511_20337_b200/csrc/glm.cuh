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
// First version of this path: one thread per zone and direction, both faces of the zone solved by the
// thread itself (every interface is solved twice; loads are x-contiguous in every direction), one launch per
// direction, an elementwise combine.  It is correct and measured, not yet fused like the CT path.
#pragma once
#include "kernels.cuh"

namespace pluto {

constexpr double kGlmCr = 0.18;      // c_p^2 / c_h of [43]

// rotated primitives of one zone for a sweep along DIR: rho, u, v, w, B_t1, B_t2, p, B_n, psi
template <int DIR>
__device__ __forceinline__ void glm_prims(const Grid &g, const double *__restrict__ S, const double *__restrict__ psi,
                                          long long c, double q[9], bool &bad)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const long long sa = g.sa;
    const double rho = S[c], En = S[4 * sa + c];
    const double m[3] = { S[sa + c], S[2 * sa + c], S[3 * sa + c] };
    const double B[3] = { S[5 * sa + c], S[6 * sa + c], S[7 * sa + c] };
    const double ir = rcp_fast(rho);
    const double v[3] = { __dmul_rn(m[0], ir), __dmul_rn(m[1], ir), __dmul_rn(m[2], ir) };
    const double p = __dmul_rn(g.gamma - 1.0, fma(-0.5, fma(B[0], B[0], fma(B[1], B[1], B[2] * B[2])),
                                                  fma(-0.5, fma(m[0], v[0], fma(m[1], v[1], m[2] * v[2])), En)));
    q[0] = rho; q[1] = v[DIR]; q[2] = v[T1]; q[3] = v[T2]; q[4] = B[T1]; q[5] = B[T2]; q[6] = p; q[7] = B[DIR];
    q[8] = psi[c];
    bad = unphysical(rho) || unphysical(p);
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
template <int DIR, int LIM, bool FIRST>
__global__ void __launch_bounds__(128)
k_glm_sweep(Grid g, const double *__restrict__ Sin, const double *__restrict__ psin, double *Sout, double *psout,
            StepParams *P)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.n[0]) return;
    const long long sa = g.sa, st = g.st[DIR], c = g.at(i, j, k);
    const double ch = P->glm_ch, dtdx = P->dtdx[DIR];
    double q[5][9];
    bool bad, mybad = false;
#pragma unroll
    for (int m = 0; m < 5; m++) {
        glm_prims<DIR>(g, Sin, psin, c + (m - 2) * st, q[m], bad);
        if (m == 2) mybad = bad;
    }
    if (mybad) P->err = 1;
    // faces of the cells c-1, c, c+1 (Eq. 6; R4): lo on the lower face, hi on the upper face
    double Ll[9], Rl[9], Lu[9], Ru[9];
#pragma unroll
    for (int v = 0; v < 9; v++) {
        double lo, hi;
        plm_faces<LIM>(q[1][v], q[1][v] - q[0][v], q[2][v] - q[1][v], lo, Ll[v]);      // cell c-1: its upper face value
        plm_faces<LIM>(q[2][v], q[2][v] - q[1][v], q[3][v] - q[2][v], Rl[v], Lu[v]);   // cell c
        plm_faces<LIM>(q[3][v], q[3][v] - q[2][v], q[4][v] - q[3][v], Ru[v], hi);      // cell c+1: its lower face value
    }
    double fl[9], fu[9];
    glm_face_flux(Ll, Rl, ch, g.gamma, g.igm1, fl);
    glm_face_flux(Lu, Ru, ch, g.gamma, g.igm1, fu);
    // rotated flux (rho, m_n, m_t1, m_t2, B_t1, B_t2, E, B_n, psi) -> state arrays
    const double *base = FIRST ? Sin : Sout;
    const double *pbase = FIRST ? psin : psout;
    Sout[c] = fma(-dtdx, fu[0] - fl[0], base[c]);
    Sout[(1 + DIR) * sa + c] = fma(-dtdx, fu[1] - fl[1], base[(1 + DIR) * sa + c]);
    Sout[(1 + T1) * sa + c] = fma(-dtdx, fu[2] - fl[2], base[(1 + T1) * sa + c]);
    Sout[(1 + T2) * sa + c] = fma(-dtdx, fu[3] - fl[3], base[(1 + T2) * sa + c]);
    Sout[4 * sa + c] = fma(-dtdx, fu[6] - fl[6], base[4 * sa + c]);
    Sout[(5 + DIR) * sa + c] = fma(-dtdx, fu[7] - fl[7], base[(5 + DIR) * sa + c]);
    Sout[(5 + T1) * sa + c] = fma(-dtdx, fu[4] - fl[4], base[(5 + T1) * sa + c]);
    Sout[(5 + T2) * sa + c] = fma(-dtdx, fu[5] - fl[5], base[(5 + T2) * sa + c]);
    psout[c] = fma(-dtdx, fu[8] - fl[8], pbase[c]);
}

// Runge-Kutta combine of the nine arrays (a7), out <- wn * S^n + ws * S~ with S~ = Euler(S) in scratch arrays
// (out may be S^n itself: in place), and, at the end of a step, the exact damping of psi
// (glm_damp = exp(-dt c_h / c_r) from the device scalars)
__global__ void __launch_bounds__(128)
k_glm_combine(Grid g, double *Sout, double *psout, const double *Sn, const double *psn,
              const double *__restrict__ St, const double *__restrict__ pst,
              double wn, double ws, int do_damp, const StepParams *__restrict__ P)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.n[0]) return;
    const long long sa = g.sa, c = g.at(i, j, k);
#pragma unroll
    for (int v = 0; v < 8; v++) Sout[v * sa + c] = fma(wn, Sn[v * sa + c], ws * St[v * sa + c]);
    double ps = fma(wn, psn[c], ws * pst[c]);
    if (do_damp) ps *= P->glm_damp;
    psout[c] = ps;
}

} // namespace pluto
