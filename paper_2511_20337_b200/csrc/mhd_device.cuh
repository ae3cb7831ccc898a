// mhd_device.cuh -- per-zone / per-interface fp64 device arithmetic of the MHD step.
//
//   prim_from_cons : Eq. 7
//   plm_slope      : limited slope for Eq. 6, minmod / MC (reading R4)
//   hlld           : HLLD flux in the rotated frame (Eq. 8; [56] PAPER.md:649; R5)
//                    + the continuous upwind weight used by CT (R6)
#pragma once
#include <cuda_runtime.h>

namespace pluto {

constexpr double kTheta = 1e-3;   // R6: |mass flux| >= theta * f_ref is fully upwinded
constexpr double kDegen = 1e-8;   // R5: guard of the star-state denominator

// ---------------------------------------------------------------- fp64 reciprocal / square root
// IEEE division and sqrt cost ~9 fp64-pipe instructions each plus range checks and a slow-path call;
// HLLD needs 9 reciprocals and 6 square roots per interface, about half of its arithmetic.  These
// versions start from the hardware seed (MUFU.RCP64H / MUFU.RSQ64H, relative error <= 2^-22) and
// refine it with a third-order / two second-order steps: results are within ~1 ulp of the IEEE
// value for normal, finite, positive-range arguments, which is all this path produces (the error
// flag catches non-positive density / pressure).  No denormal, zero or infinity handling.
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);          // e = 1 - x y,  |e| <= 2^-22
    e = fma(e, e, e);                    // e + e^2
    return fma(y, e, y);                 // y (1 + e + e^2): error ~ e^3
}

// s = sqrt(x), returns also r = 1/sqrt(x); x > 0
__device__ __forceinline__ void sqrt_rsqrt_fast(double x, double &s, double &r)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double g = x * y, h = 0.5 * y;       // g -> sqrt(x), h -> 1/(2 sqrt(x))
    double e = fma(-g, h, 0.5);
    g = fma(g, e, g); h = fma(h, e, h);
    e = fma(-g, h, 0.5);
    s = fma(g, e, g);
    r = 2.0 * fma(h, e, h);
}

__device__ __forceinline__ double sqrt_fast(double x)
{
    double s, r;
    sqrt_rsqrt_fast(x, s, r);
    return s;
}

// sqrt that tolerates x == 0 (the discriminant of the fast speed can vanish)
__device__ __forceinline__ double sqrt_fast0(double x)
{
    double s = sqrt_fast(fmax(x, 1e-300));
    return x > 0.0 ? s : 0.0;
}

template <int LIM>
__device__ __forceinline__ double plm_slope(double dm, double dp)
{
    if (LIM == 0) {
        double s = fabs(dm) < fabs(dp) ? dm : dp;
        return dm * dp > 0.0 ? s : 0.0;
    } else {
        double sum = dm + dp;
        double mag = fmin(2.0 * fmin(fabs(dm), fabs(dp)), 0.5 * fabs(sum));
        double s = sum > 0.0 ? mag : -mag;
        return dm * dp > 0.0 ? s : 0.0;
    }
}

// fast magnetosonic speed from a^2*rho = gamma*p, B-normal^2 and |B|^2 (all divided by rho inside)
__device__ __forceinline__ double fast_speed(double rho, double gp, double bn2, double b2)
{
    double ir  = rcp_fast(rho);
    double a2  = gp * ir;
    double s   = a2 + b2 * ir;
    double disc = s * s - 4.0 * a2 * (bn2 * ir);
    return sqrt_fast(0.5 * (s + sqrt_fast0(disc)));
}

// One side of the Riemann fan in the rotated frame.
struct Side {
    double rho, u, v, w, By, Bz, p;     // reconstructed primitives (B-normal is shared)
};

// HLLD flux.  Output f[7] = (rho, m_n, m_t1, m_t2, B_t1, B_t2, E) flux, wgt = upwind weight.
__device__ __forceinline__ void hlld(const Side &L, const Side &R, double Bx, double gamma, double igm1,
                                     double f[7], double &wgt)
{
    const double Bx2 = Bx * Bx;

    // left / right total pressure, v.B, energy, physical flux
    double BtL2 = L.By * L.By + L.Bz * L.Bz, BtR2 = R.By * R.By + R.Bz * R.Bz;
    double pTL = L.p + 0.5 * (Bx2 + BtL2), pTR = R.p + 0.5 * (Bx2 + BtR2);
    double vBL = L.u * Bx + L.v * L.By + L.w * L.Bz;
    double vBR = R.u * Bx + R.v * R.By + R.w * R.Bz;
    double EL = L.p * igm1 + 0.5 * L.rho * (L.u * L.u + L.v * L.v + L.w * L.w) + 0.5 * (Bx2 + BtL2);
    double ER = R.p * igm1 + 0.5 * R.rho * (R.u * R.u + R.v * R.v + R.w * R.w) + 0.5 * (Bx2 + BtR2);

    double cfL = fast_speed(L.rho, gamma * L.p, Bx2, Bx2 + BtL2);
    double cfR = fast_speed(R.rho, gamma * R.p, Bx2, Bx2 + BtR2);
    double cmax = fmax(cfL, cfR);
    double SL = fmin(L.u, R.u) - cmax;
    double SR = fmax(L.u, R.u) + cmax;

    // the side the interface lies in is decided by S_M; supersonic cases fall out of the same test
    double aL = L.rho * (SL - L.u), aR = R.rho * (SR - R.u);
    double idenom = rcp_fast(aR - aL);
    double SM  = (aR * R.u - aL * L.u - pTR + pTL) * idenom;
    double pTs = (aR * pTL - aL * pTR + aL * aR * (R.u - L.u)) * idenom;

    // star states of both sides (transverse velocity and field, density, energy)
    double rsL, vsL, wsL, BysL, BzsL, EsL, vBsL;
    double rsR, vsR, wsR, BysR, BzsR, EsR, vBsR;
    {
        double dS = SL - SM, idS = rcp_fast(dS);
        double D = aL * dS - Bx2;
        rsL = aL * idS;
        if (fabs(D) <= kDegen * pTs) {
            vsL = L.v; wsL = L.w; BysL = L.By; BzsL = L.Bz;
        } else {
            double iD = rcp_fast(D);
            double cv = Bx * (SM - L.u) * iD;
            double cb = (aL * (SL - L.u) - Bx2) * iD;
            vsL = L.v - cv * L.By; wsL = L.w - cv * L.Bz;
            BysL = L.By * cb;      BzsL = L.Bz * cb;
        }
        vBsL = SM * Bx + vsL * BysL + wsL * BzsL;
        EsL = ((SL - L.u) * EL - pTL * L.u + pTs * SM + Bx * (vBL - vBsL)) * idS;
    }
    {
        double dS = SR - SM, idS = rcp_fast(dS);
        double D = aR * dS - Bx2;
        rsR = aR * idS;
        if (fabs(D) <= kDegen * pTs) {
            vsR = R.v; wsR = R.w; BysR = R.By; BzsR = R.Bz;
        } else {
            double iD = rcp_fast(D);
            double cv = Bx * (SM - R.u) * iD;
            double cb = (aR * (SR - R.u) - Bx2) * iD;
            vsR = R.v - cv * R.By; wsR = R.w - cv * R.Bz;
            BysR = R.By * cb;      BzsR = R.Bz * cb;
        }
        vBsR = SM * Bx + vsR * BysR + wsR * BzsR;
        EsR = ((SR - R.u) * ER - pTR * R.u + pTs * SM + Bx * (vBR - vBsR)) * idS;
    }

    // Alfven waves and the double-star state
    double rL, rR, irL, irR;
    sqrt_rsqrt_fast(rsL, rL, irL);
    sqrt_rsqrt_fast(rsR, rR, irR);
    double aBx = fabs(Bx);
    double SaL = SM - aBx * irL, SaR = SM + aBx * irR;
    double sig = Bx > 0.0 ? 1.0 : (Bx < 0.0 ? -1.0 : 0.0);
    double iR = rcp_fast(rL + rR);
    double vss  = (rL * vsL + rR * vsR + sig * (BysR - BysL)) * iR;
    double wss  = (rL * wsL + rR * wsR + sig * (BzsR - BzsL)) * iR;
    double Byss = (rL * BysR + rR * BysL + sig * rL * rR * (vsR - vsL)) * iR;
    double Bzss = (rL * BzsR + rR * BzsL + sig * rL * rR * (wsR - wsL)) * iR;
    double vBss = SM * Bx + vss * Byss + wss * Bzss;

    // pick the side, then the region on that side
    // (test order of R5: S_L >= 0, S_R <= 0, S*_L >= 0, S_M >= 0, S*_R > 0; S*_L <= S_M always)
    const bool supL = SL >= 0.0;
    const bool supR = !supL && SR <= 0.0;
    const bool supersonic = supL || supR;
    const bool left = supL || (!supR && SM >= 0.0);
    const bool outer = left ? (SaL >= 0.0) : !(SaR > 0.0);

    const Side &K = left ? L : R;
    double S   = left ? SL : SR;
    double Sa  = left ? SaL : SaR;
    double pT  = left ? pTL : pTR;
    double vB  = left ? vBL : vBR;
    double E   = left ? EL : ER;
    double rs  = left ? rsL : rsR;
    double vs  = left ? vsL : vsR,  ws  = left ? wsL : wsR;
    double Bys = left ? BysL : BysR, Bzs = left ? BzsL : BzsR;
    double Es  = left ? EsL : EsR,  vBs = left ? vBsL : vBsR;
    double r   = left ? rL : rR;
    double sg  = left ? -sig : sig;

    // physical flux of the chosen side (Eq. 2)
    double F0 = K.rho * K.u;
    double F1 = F0 * K.u + pT - Bx2;
    double F2 = F0 * K.v - Bx * K.By;
    double F3 = F0 * K.w - Bx * K.Bz;
    double F5 = K.By * K.u - Bx * K.v;
    double F6 = K.Bz * K.u - Bx * K.w;
    double F7 = (E + pT) * K.u - Bx * vB;

    if (!supersonic) {
        // conserved vectors U (chosen side), U*, U**
        double U0 = K.rho, U1 = K.rho * K.u, U2 = K.rho * K.v, U3 = K.rho * K.w;
        double Us1 = rs * SM, Us2 = rs * vs, Us3 = rs * ws;
        if (outer) {
            F0 += S * (rs - U0);   F1 += S * (Us1 - U1);  F2 += S * (Us2 - U2);  F3 += S * (Us3 - U3);
            F5 += S * (Bys - K.By); F6 += S * (Bzs - K.Bz); F7 += S * (Es - E);
        } else {
            double Ess = Es + sg * r * (vBs - vBss);
            double c1 = Sa - S;     // F + Sa*U** - (Sa - S)*U* - S*U
            F0 += Sa * rs - c1 * rs - S * U0;
            F1 += Sa * (rs * SM) - c1 * Us1 - S * U1;
            F2 += Sa * (rs * vss) - c1 * Us2 - S * U2;
            F3 += Sa * (rs * wss) - c1 * Us3 - S * U3;
            F5 += Sa * Byss - c1 * Bys - S * K.By;
            F6 += Sa * Bzss - c1 * Bzs - S * K.Bz;
            F7 += Sa * Ess - c1 * Es - S * E;
        }
    }
    f[0] = F0; f[1] = F1; f[2] = F2; f[3] = F3; f[4] = F5; f[5] = F6; f[6] = F7;

    double fref = 0.25 * (L.rho + R.rho) * (SR - SL);
    double wv = 0.5 + 0.5 * F0 * rcp_fast(kTheta * fref);
    wgt = fmin(fmax(wv, 0.0), 1.0);
}

} // namespace pluto
