// mhd_device.cuh -- per-zone / per-interface fp64 device arithmetic of the MHD step.
//
//   prim_from_cons : Eq. 7
//   plm_slope      : limited slope for Eq. 6, minmod / MC (reading R4)
//   hlld           : HLLD flux in the rotated frame (Eq. 8; [56] PAPER.md:649; R5)
//                    + the continuous upwind weight used by CT (R6)
//
// Rounding discipline.  These functions are inlined at several sites (the first cells of a march segment
// and its running loop, the two unrolled copies of a loop body), and the compiler is free to contract
// a * b + c into an FMA differently at each site.  Wherever a product feeds an addition the choice is
// therefore written out -- fma() or __dmul_rn() (which is never contracted) -- so that a flux is the same
// bits wherever it is evaluated and a run does not depend on how the marches are cut into segments or the
// box into slabs.  Products that only feed other products, selects or comparisons are left plain.
#pragma once
#include <cuda_runtime.h>

namespace pluto {

constexpr double kTheta = 1e-3;   // R6: |mass flux| >= theta * f_ref is fully upwinded
constexpr double kDegen = 1e-8;   // R5: guard of the star-state denominator

// ---------------------------------------------------------------- fp64 reciprocal / square root
// IEEE division and sqrt cost ~9 fp64-pipe instructions each plus range checks and a slow-path call;
// HLLD needs 9 reciprocals and 5 square roots per interface, about a third of its arithmetic.  These
// versions start from the hardware seed (MUFU.RCP64H / MUFU.RSQ64H, relative error <= 2^-22) and
// refine it with a third-order step / a second-order step plus a residual correction: results are
// within ~1 ulp of the IEEE value for normal, finite, positive-range arguments, which is all this path
// produces (the error flag catches non-positive density / pressure).  No denormal, zero or infinity
// handling.
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);          // e = 1 - x y,  |e| <= 2^-22
    e = fma(e, e, e);                    // e + e^2
    return fma(y, e, y);                 // y (1 + e + e^2): error ~ e^3
}

// sqrt(x), x > 0: one coupled Newton step on (g, h) -> (sqrt x, 1 / (2 sqrt x)) takes the seed's relative
// error d to g (1 - 3/2 d^2); the exact residual x - g^2 (one fma) times the unrefined h then cancels
// the d^2 term: g (1 + 3/2 d^3), below half an ulp before the final rounding.  Six fp64-pipe instructions.
__device__ __forceinline__ double sqrt_fast(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double g = x * y, h = 0.5 * y;
    const double e = fma(-g, h, 0.5);
    g = fma(g, e, g);
    return fma(fma(-g, g, x), h, g);
}

// max / min of two numbers by one comparison and a select (three instructions).  fmax() / fmin() also
// quiet NaNs, seven instructions for the IEEE rule, and the compiler turns a > b ? a : b back into them when
// b is a constant: hence PTX.  No NaN reaches these on a physical state, and an unphysical one is reported
// by the sweeps' own check.  A NaN in `a` returns b.
__device__ __forceinline__ double max_sel(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.gt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}
__device__ __forceinline__ double min_sel(double a, double b)
{
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.lt.f64 p, %1, %2;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b));
    return r;
}

// Limited slope (R4).  The sign test dm * dp > 0 is taken on the sign bits (integer pipe) instead
// of a DMUL + DSETP: identical unless dm * dp underflows, where the slope is < 1e-154 anyway.
template <int LIM>
__device__ __forceinline__ double plm_slope(double dm, double dp)
{
    const bool same = (__double2hiint(dm) ^ __double2hiint(dp)) >= 0;
    if (LIM == 0) {
        double s = fabs(dm) < fabs(dp) ? dm : dp;     // a zero difference is returned as itself
        return same ? s : 0.0;
    } else {
        double sum = dm + dp;
        double mag = fmin(2.0 * fmin(fabs(dm), fabs(dp)), 0.5 * fabs(sum));
        return same ? copysign(mag, dm) : 0.0;        // same sign: sign(dm + dp) = sign(dm)
    }
}

// Interface values of a cell with value q and one-sided differences dm, dp (Eq. 6):
// lo = q - s/2 on its lower face, hi = q + s/2 on its upper face.  The zero-slope case multiplies by
// a selected half-weight (0.5 or 0) instead of selecting the slope: one select fewer per variable.
template <int LIM>
__device__ __forceinline__ void plm_faces(double q, double dm, double dp, double &lo, double &hi)
{
    const bool same = (__double2hiint(dm) ^ __double2hiint(dp)) >= 0;
    const double h = __hiloint2double(same ? 0x3fe00000 : 0, 0);      // 0.5 or 0.0
    double s;
    if (LIM == 0) {
        s = fabs(dm) < fabs(dp) ? dm : dp;
    } else {
        double sum = dm + dp;
        s = copysign(fmin(2.0 * fmin(fabs(dm), fabs(dp)), 0.5 * fabs(sum)), dm);
    }
    lo = fma(-h, s, q);
    hi = fma(h, s, q);
}

// WENO-Z values on both faces of the centre cell c of the stencil (a, b, c, d, e) ([51] named at
// PAPER.md:100,260; reading R18: candidate values q_k, Jiang-Shu smoothness indicators beta_k,
// tau5 = |beta0 - beta2|, alpha_k = d_k (1 + tau5 / (beta_k + 1e-40)), d = (1/10, 6/10, 3/10)).
// The same weights and values, arranged for the fp64 pipe (65 instructions for both faces, 82 before):
//  - everything is formed from the four differences d1..d4 of neighbouring cells:
//    6 q_k = 6 c + delta_k, so the face value is  c + sum(alpha_k delta_k) / (6 sum(alpha_k));
//  - the indicators are carried as 4 beta_k = 13/3 a_k^2 + b_k^2 with 4 eps (scaling by four is exact, the
//    quotient tau5 / (beta_k + eps) is the same number);
//  - the normalised weights do not change when every alpha_k is multiplied by the common positive factor
//    P0 P1 P2, P_k = 4 (beta_k + eps):  alpha_k -> d_k (P_k + 4 tau5) P_l P_m  -- products instead of three
//    reciprocals (|q| < 1e50 keeps them inside the fp64 range);
//  - the lower-face value is the same formula on the mirrored stencil: beta_0 and beta_2 swap, beta_1 and
//    tau5 are unchanged, so the indicators and the three products are formed once for both faces.
// Every product that feeds a sum is an explicit fma / __dmul_rn (see the header: same bits at every site).
__device__ __forceinline__ void wenoz_faces(double a, double b, double c, double d, double e, double &lo, double &hi)
{
    const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
    const double a0 = d2 - d1, b0 = fma(3.0, d2, -d1);          // a - 2b + c,  a - 4b + 3c
    const double a1 = d3 - d2, b1 = d2 + d3;                    // b - 2c + d,  -(b - d)
    const double a2 = d4 - d3, b2 = fma(-3.0, d3, d4);          // c - 2d + e,  3c - 4d + e
    const double P0 = fma(13.0 / 3.0 * a0, a0, __dmul_rn(b0, b0)) + 4e-40;
    const double P1 = fma(13.0 / 3.0 * a1, a1, __dmul_rn(b1, b1)) + 4e-40;
    const double P2 = fma(13.0 / 3.0 * a2, a2, __dmul_rn(b2, b2)) + 4e-40;
    const double tau = fabs(P0 - P2);
    const double W0 = (P0 + tau) * (P1 * P2), W1 = (P1 + tau) * (P0 * P2), W2 = (P2 + tau) * (P0 * P1);
    const double m1 = 0.6 * W1;
    // upper face: stencils (a,b,c), (b,c,d), (c,d,e) with d = (0.1, 0.6, 0.3)
    {
        const double al0 = 0.1 * W0, al2 = 0.3 * W2;
        const double num = fma(al0, fma(5.0, d2, -2.0 * d1), fma(m1, fma(2.0, d3, d2), __dmul_rn(al2, fma(4.0, d3, -d4))));
        hi = fma(num, rcp_fast(6.0 * (al0 + m1 + al2)), c);
    }
    // lower face: the mirrored stencils (e,d,c), (d,c,b), (c,b,a)
    {
        const double al0 = 0.1 * W2, al2 = 0.3 * W0;
        const double num = fma(al0, fma(-5.0, d3, 2.0 * d4), fma(m1, -fma(2.0, d2, d3), __dmul_rn(al2, fma(-4.0, d2, d1))));
        lo = fma(num, rcp_fast(6.0 * (al0 + m1 + al2)), c);
    }
}

// The upper-face value alone (the lower-face value of a cell is this on the mirrored stencil): same arithmetic
// as the upper face of wenoz_faces, 49 fp64 instructions.  Used where the two faces of a cell are wanted by
// different threads (the edge reconstruction of uct.cuh).
__device__ __forceinline__ double wenoz_upper(double a, double b, double c, double d, double e)
{
    const double d1 = b - a, d2 = c - b, d3 = d - c, d4 = e - d;
    const double a0 = d2 - d1, b0 = fma(3.0, d2, -d1);
    const double a1 = d3 - d2, b1 = d2 + d3;
    const double a2 = d4 - d3, b2 = fma(-3.0, d3, d4);
    const double P0 = fma(13.0 / 3.0 * a0, a0, __dmul_rn(b0, b0)) + 4e-40;
    const double P1 = fma(13.0 / 3.0 * a1, a1, __dmul_rn(b1, b1)) + 4e-40;
    const double P2 = fma(13.0 / 3.0 * a2, a2, __dmul_rn(b2, b2)) + 4e-40;
    const double tau = fabs(P0 - P2);
    const double al0 = 0.1 * ((P0 + tau) * (P1 * P2)), m1 = 0.6 * ((P1 + tau) * (P0 * P2)), al2 = 0.3 * ((P2 + tau) * (P0 * P1));
    const double num = fma(al0, fma(5.0, d2, -2.0 * d1), fma(m1, fma(2.0, d3, d2), __dmul_rn(al2, fma(4.0, d3, -d4))));
    return fma(num, rcp_fast(6.0 * (al0 + m1 + al2)), c);
}

// Interface values of the centre cell from its five-cell stencil: LIM 0/1 = PLM with minmod / MC
// (uses the inner three cells), LIM 2 = WENO-Z.  lo on the lower face, hi on the upper face.
template <int LIM>
__device__ __forceinline__ void recon_faces(double qm2, double qm1, double q0, double qp1, double qp2,
                                            double &lo, double &hi)
{
    if (LIM == 2) wenoz_faces(qm2, qm1, q0, qp1, qp2, lo, hi);
    else plm_faces<LIM == 2 ? 0 : LIM>(q0, q0 - qm1, qp1 - q0, lo, hi);
}

// rho or p is unphysical: not a positive, finite, normal number (sign / exponent test on the high word)
__device__ __forceinline__ bool unphysical(double x)
{
    return (unsigned)(__double2hiint(x) - 0x00100000) >= 0x7fe00000u;
}

// square of the fast magnetosonic speed from gp = gamma * p, B-normal^2 and |B|^2:
// c_f^2 = s/2 + sqrt((s/2)^2 - a^2 b_n^2 / rho),  s = a^2 + B^2 / rho  (the halved form of
// (s + sqrt(s^2 - 4 a^2 b_n^2/rho)) / 2: scaling by two is exact, so the roundings are the same)
__device__ __forceinline__ double fast_speed2(double rho, double gp, double bn2, double b2)
{
    const double ir = rcp_fast(rho);
    const double a2 = gp * ir;
    const double h  = 0.5 * fma(b2, ir, a2);
    const double disc = fma(h, h, -(a2 * (bn2 * ir)));
    return h + sqrt_fast(max_sel(disc, 1e-300));        // max(0, disc) of R5 up to 1e-150
}

// One side of the Riemann fan in the rotated frame.
struct Side {
    double rho, u, v, w, By, Bz, p;     // reconstructed primitives (B-normal is shared)
};

// HLLD flux (R5).  Output f[7] = (rho, m_n, m_t1, m_t2, B_t1, B_t2, E) flux, wgt = upwind weight (R6).
//
// The interface state is picked first -- the side by S_M, then U* or U** by the Alfven wave -- and the
// flux is evaluated from that state, F = F(rho, S_M, v, w, By, Bz, E; pT*).  The HLLD states satisfy
// the jump conditions S (U_b - U_a) = F_b - F_a with exactly these fluxes, so this equals the
// jump form F_K + S_K (U* - U_K) [+ S* (U** - U*)] of the HLLD paper up to rounding (in the guarded
// degenerate case the two differ by < 1e-8 pT* B_t |S_M - u|, second order small).  Only the chosen
// side's energy chain is computed.  Supersonic fans take the rarely executed branch at the end.
//
// UCT = true also returns what the UCT-HLLD EMF average ([47] named at PAPER.md:271; reading R19) takes from the
// interface: uct[5] = a^L, d^L, d^R and the transverse velocities a^L v^L + a^R v^R, a^L w^L + a^R w^R, where
//     F[B_t] = a^L (u B_t)^L + a^R (u B_t)^R - (d^R B_t^R - d^L B_t^L) - B_n (a^L v_t^L + a^R v_t^R)
// is the (unique) decomposition of the HLLD induction flux that is linear in the four transverse inputs:
//     chi^s = (u^s - S_M)(S_s - S_M) / (S*_s + S_s - 2 S_M),   nu^s = (S*_s + S_s) / (|S*_s| + |S_s|),
//     nu* = (S*_R + S*_L) / (|S*_R| + |S*_L|)  (0 when both Alfven speeds vanish),
//     a^L = (1 + nu*)/2,  d^s = (nu^s - nu*) chi^s / 2 + (|S*_s| - nu* S*_s) / 2.
template <bool UCT>
__device__ __forceinline__ void hlld_t(const Side &L, const Side &R, double Bx, double gamma, double igm1,
                                       double f[7], double &wgt, double uct[5])
{
    const double Bx2 = __dmul_rn(Bx, Bx);
    const double B2L = Bx2 + fma(L.By, L.By, L.Bz * L.Bz), B2R = Bx2 + fma(R.By, R.By, R.Bz * R.Bz);
    const double pTL = fma(0.5, B2L, L.p), pTR = fma(0.5, B2R, R.p);

    const double cmax = sqrt_fast(max_sel(fast_speed2(L.rho, gamma * L.p, Bx2, B2L),
                                          fast_speed2(R.rho, gamma * R.p, Bx2, B2R)));
    const double SL = min_sel(L.u, R.u) - cmax, SR = max_sel(L.u, R.u) + cmax;
    const double dL = SL - L.u, dR = SR - R.u;              // S_a - u_a
    const double aL = __dmul_rn(L.rho, dL), aR = __dmul_rn(R.rho, dR);
    const double idenom = rcp_fast(aR - aL);
    const double SM  = __dmul_rn(fma(aR, R.u, fma(-aL, L.u, pTL - pTR)), idenom);
    const double pTs = __dmul_rn(fma(aR, pTL, fma(-aL, pTR, aL * aR * (R.u - L.u))), idenom);
    const double guard = kDegen * pTs;

    // star states: density and the transverse velocity / field of both sides
    double rsL, vsL, wsL, BysL, BzsL, idSL;
    double rsR, vsR, wsR, BysR, BzsR, idSR;
    {
        const double dS = SL - SM, D = fma(aL, dS, -Bx2);
        idSL = rcp_fast(dS);
        rsL = __dmul_rn(aL, idSL);
        // (S_M - u)/D, zero in the guarded degenerate case: then v* = v, B_t* = B_t (R5)
        const double m = fabs(D) <= guard ? 0.0 : (dL - dS) * rcp_fast(D);
        const double cv = Bx * m, cb = aL * m;                      // B_t*/B_t = 1 + a (S_M - u)/D
        vsL = fma(-cv, L.By, L.v); wsL = fma(-cv, L.Bz, L.w);
        BysL = fma(L.By, cb, L.By); BzsL = fma(L.Bz, cb, L.Bz);
    }
    {
        const double dS = SR - SM, D = fma(aR, dS, -Bx2);
        idSR = rcp_fast(dS);
        rsR = __dmul_rn(aR, idSR);
        const double m = fabs(D) <= guard ? 0.0 : (dR - dS) * rcp_fast(D);
        const double cv = Bx * m, cb = aR * m;
        vsR = fma(-cv, R.By, R.v); wsR = fma(-cv, R.Bz, R.w);
        BysR = fma(R.By, cb, R.By); BzsR = fma(R.Bz, cb, R.Bz);
    }

    // double-star state (common to both sides apart from density and energy)
    const double rL = sqrt_fast(rsL), rR = sqrt_fast(rsR);
    // sigma = sign(Bx); for Bx = 0 the double-star state is never selected (outer is always true)
    const double sig = copysign(1.0, Bx);
    const double iR = rcp_fast(rL + rR);
    const double srr = sig * rL * rR;
    const double vss  = fma(sig, BysR - BysL, fma(rL, vsL, rR * vsR)) * iR;
    const double wss  = fma(sig, BzsR - BzsL, fma(rL, wsL, rR * wsR)) * iR;
    const double Byss = fma(srr, vsR - vsL, fma(rL, BysR, rR * BysL)) * iR;
    const double Bzss = fma(srr, wsR - wsL, fma(rL, BzsR, rR * BzsL)) * iR;
    const double SMBx = __dmul_rn(SM, Bx);
    const double vBss = fma(vss, Byss, fma(wss, Bzss, SMBx));

    // the side the interface lies in (test order of R5: ..., S*_L >= 0, S_M >= 0, S*_R > 0), and
    // whether it lies outside the Alfven wave of that side:  S*_L = S_M - |Bx|/rL >= 0, S*_R = S_M + |Bx|/rR <= 0
    const bool left = SM >= 0.0;
    const double rho = left ? L.rho : R.rho, u = left ? L.u : R.u, v = left ? L.v : R.v, w = left ? L.w : R.w;
    const double By = left ? L.By : R.By, Bz = left ? L.Bz : R.Bz, p = left ? L.p : R.p;
    const double B2 = left ? B2L : B2R, pT = left ? pTL : pTR, d = left ? dL : dR, idS = left ? idSL : idSR;
    const double rs = left ? rsL : rsR, r = left ? rL : rR;
    const double vs = left ? vsL : vsR, ws = left ? wsL : wsR, Bys = left ? BysL : BysR, Bzs = left ? BzsL : BzsR;
    const bool outer = fabs(SM) * r >= fabs(Bx);

    // energy of the chosen side: U, U*, U**
    const double E  = fma(p, igm1, 0.5 * fma(rho, fma(u, u, fma(v, v, w * w)), B2));
    const double vB = fma(u, Bx, fma(v, By, w * Bz));
    const double vBs = fma(vs, Bys, fma(ws, Bzs, SMBx));
    const double Es = __dmul_rn(fma(d, E, -pT * u) + fma(pTs, SM, Bx * (vB - vBs)), idS);
    const double sr = left ? -sig * r : sig * r;
    const double Ess = fma(sr, vBs - vBss, Es);

    double rho_f = rs, uf = SM, pf = pTs;
    double vf = outer ? vs : vss, wf = outer ? ws : wss, Byf = outer ? Bys : Byss, Bzf = outer ? Bzs : Bzss;
    double Ef = outer ? Es : Ess, vBf = outer ? vBs : vBss;
    if (UCT) {
        const double aBx = fabs(Bx);
        const double SaL = fma(-aBx, rcp_fast(rL), SM), SaR = fma(aBx, rcp_fast(rR), SM);     // Alfven speeds S*_L, S*_R
        const double chiL = (L.u - SM) * (SL - SM) * rcp_fast((SaL + SL) - 2.0 * SM);
        const double chiR = (R.u - SM) * (SR - SM) * rcp_fast((SaR + SR) - 2.0 * SM);
        const double nuL = (SaL + SL) * rcp_fast(fabs(SaL) + fabs(SL));
        const double nuR = (SaR + SR) * rcp_fast(fabs(SaR) + fabs(SR));
        const double den = fabs(SaR) + fabs(SaL);
        const double nus = den > 0.0 ? (SaR + SaL) * rcp_fast(den) : 0.0;
        const double al = fma(0.5, nus, 0.5), ar = fma(-0.5, nus, 0.5);
        uct[0] = al;
        uct[1] = fma(0.5 * (nuL - nus), chiL, 0.5 * fma(-nus, SaL, fabs(SaL)));
        uct[2] = fma(0.5 * (nuR - nus), chiR, 0.5 * fma(-nus, SaR, fabs(SaR)));
        uct[3] = fma(al, L.v, ar * R.v);
        uct[4] = fma(al, L.w, ar * R.w);
    }
    if (__builtin_expect(SL >= 0.0 || SR <= 0.0, 0)) {          // one-sided fan: the upwind physical flux (Eq. 2)
        const bool sl = SL >= 0.0;
        if (UCT) { uct[0] = sl ? 1.0 : 0.0; uct[1] = 0.0; uct[2] = 0.0; uct[3] = sl ? L.v : R.v; uct[4] = sl ? L.w : R.w; }
        rho_f = sl ? L.rho : R.rho; uf = sl ? L.u : R.u; vf = sl ? L.v : R.v; wf = sl ? L.w : R.w;
        Byf = sl ? L.By : R.By; Bzf = sl ? L.Bz : R.Bz; pf = sl ? pTL : pTR;
        {
            const double pp = sl ? L.p : R.p, bb = sl ? B2L : B2R;
            Ef = fma(pp, igm1, 0.5 * fma(rho_f, fma(uf, uf, fma(vf, vf, wf * wf)), bb));
        }
        vBf = fma(uf, Bx, fma(vf, Byf, wf * Bzf));
    }
    const double F0 = __dmul_rn(rho_f, uf);      // a rounded product: the same bits for both cells sharing the face
    f[0] = F0;
    f[1] = fma(F0, uf, pf - Bx2);
    f[2] = fma(F0, vf, -Bx * Byf);
    f[3] = fma(F0, wf, -Bx * Bzf);
    f[4] = fma(Byf, uf, -Bx * vf);
    f[5] = fma(Bzf, uf, -Bx * wf);
    f[6] = fma(Ef + pf, uf, -Bx * vBf);

    // R6: w = clamp(1/2 + F[rho] / (2 theta f_ref)), f_ref = (rho_L + rho_R)(S_R - S_L) / 4
    const double wv = fma(F0, rcp_fast((0.5 * kTheta) * ((L.rho + R.rho) * (SR - SL))), 0.5);
    wgt = min_sel(max_sel(wv, 0.0), 1.0);
}

__device__ __forceinline__ void hlld(const Side &L, const Side &R, double Bx, double gamma, double igm1,
                                     double f[7], double &wgt)
{
    double none[5];
    hlld_t<false>(L, R, Bx, gamma, igm1, f, wgt, none);
}

} // namespace pluto
