// kernels.cuh -- CUDA kernels of the MHD step (sm_100a), baseline multi-kernel form.
// One thread per zone / face / edge, x fastest so every warp access is a contiguous 256 B row.
#pragma once
#include "grid.h"
#include "mhd_device.cuh"

namespace pluto {

struct Box { int lo[3], hi[3]; };   // inclusive lo, exclusive hi

__device__ __forceinline__ bool thread_zone(const Box &b, int &i, int &j, int &k)
{
    i = b.lo[0] + blockIdx.x * blockDim.x + threadIdx.x;
    j = b.lo[1] + blockIdx.y;
    k = b.lo[2] + blockIdx.z;
    return i < b.hi[0];
}

// ---------------------------------------------------------------- periodic ghost fill (a1)
// Fill the ghost layers of `narr` consecutive arrays along AXIS: index g in [-ng,0) <- g + n,
// g in [n, n+ng] <- g - n (cells and faces alike; face n duplicates face 0).  Launched x, then y,
// then z over the full padded extent of the other axes so edges and corners come out right
// (the paper exchanges with diagonal neighbours for the same reason).
template <int AXIS>
__global__ void k_ghost(Grid g, double *__restrict__ base, int narr)
{
    // thread x runs over padded x (AXIS != 0) or over the 2*ng+1 ghost indices (AXIS == 0)
    const int nghost = 2 * g.ng + 1;
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    int p[3];
    if (AXIS == 0) {
        if (t >= nghost) return;
        p[0] = t; p[1] = blockIdx.y; p[2] = blockIdx.z % g.tot[2];
    } else {
        if (t >= g.tot[0]) return;
        p[0] = t;
        if (AXIS == 1) { p[1] = blockIdx.y; p[2] = blockIdx.z % g.tot[2]; }
        else           { p[1] = blockIdx.y; p[2] = blockIdx.z % nghost; }
    }
    int arr = (AXIS == 2) ? blockIdx.z / nghost : blockIdx.z / g.tot[2];
    if (arr >= narr) return;
    // ghost slot -> logical index along AXIS
    int slot = p[AXIS];
    int gi = slot < g.ng ? slot - g.ng : g.n[AXIS] + (slot - g.ng);
    int src = gi < 0 ? gi + g.n[AXIS] : gi - g.n[AXIS];
    long long o[3] = { p[0], p[1], p[2] };
    long long dst_idx, src_idx;
    o[AXIS] = gi + g.off[AXIS];
    dst_idx = o[2] * g.st[2] + o[1] * g.st[1] + o[0];
    o[AXIS] = src + g.off[AXIS];
    src_idx = o[2] * g.st[2] + o[1] * g.st[1] + o[0];
    double *a = base + (long long)arr * g.sa;
    a[dst_idx] = a[src_idx];
}

// ---------------------------------------------------------------- cons -> prim (a2), Eq. 7
__global__ void k_prim(Grid g, Box box, const double *__restrict__ U, double *__restrict__ V, StepParams *P)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    long long c = g.at(i, j, k);
    double rho = U[c], mx = U[g.sa + c], my = U[2 * g.sa + c], mz = U[3 * g.sa + c];
    double Bx = U[4 * g.sa + c], By = U[5 * g.sa + c], Bz = U[6 * g.sa + c], E = U[7 * g.sa + c];
    double vx = mx / rho, vy = my / rho, vz = mz / rho;
    double p = (g.gamma - 1.0) * (E - 0.5 * (mx * vx + my * vy + mz * vz) - 0.5 * (Bx * Bx + By * By + Bz * Bz));
    V[c] = rho; V[g.sa + c] = vx; V[2 * g.sa + c] = vy; V[3 * g.sa + c] = vz;
    V[4 * g.sa + c] = Bx; V[5 * g.sa + c] = By; V[6 * g.sa + c] = Bz; V[7 * g.sa + c] = p;
    if (!(rho > 0.0) || !(p > 0.0) || isinf(rho) || isinf(p)) P->err = 1;
}

// ---------------------------------------------------------------- PLM + HLLD (a3, a4)
// Thread = lower DIR-face of cell (i,j,k).  Reads the 7 reconstructed primitives of the four
// cells c-2 .. c+1 along DIR and the face-normal field; writes the 5 hydro flux components in lab
// order, the two induction fluxes CT needs and the upwind weight.
template <int DIR, int LIM>
__global__ void __launch_bounds__(128)
k_flux(Grid g, Box box, const double *__restrict__ V, const double *__restrict__ bn, double *__restrict__ F)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const long long c = g.at(i, j, k), s = g.st[DIR], sa = g.sa;
    const int comp[7] = { 0, 1 + DIR, 1 + T1, 1 + T2, 4 + T1, 4 + T2, 7 };
    double l[7], r[7];
#pragma unroll
    for (int q = 0; q < 7; q++) {
        const double *Q = V + comp[q] * sa + c;
        double qm2 = Q[-2 * s], qm1 = Q[-s], q0 = Q[0], qp1 = Q[s];
        double d0 = q0 - qm1;
        l[q] = qm1 + 0.5 * plm_slope<LIM>(qm1 - qm2, d0);
        r[q] = q0 - 0.5 * plm_slope<LIM>(d0, qp1 - q0);
    }
    Side L = { l[0], l[1], l[2], l[3], l[4], l[5], l[6] };
    Side R = { r[0], r[1], r[2], r[3], r[4], r[5], r[6] };
    double f[7], w;
    hlld(L, R, bn[c], g.gamma, f, w);
    F[c] = f[0];
    F[(1 + DIR) * sa + c] = f[1];
    F[(1 + T1) * sa + c] = f[2];
    F[(1 + T2) * sa + c] = f[3];
    F[4 * sa + c] = f[6];
    F[5 * sa + c] = f[4];
    F[6 * sa + c] = f[5];
    F[7 * sa + c] = w;
}

// ---------------------------------------------------------------- flux-difference update (a5) [+ RK2 combine (a7)]
// Uout = Uin - sum_d dt/dx_d (F_d(+) - F_d(-)) for rho, m, E (and B_z in 2D, which has no faces).
// COMBINE: Uout <- (Uout + that)/2 in place (Uout holds U^n) -- Eq. 5's form with R3.
template <bool COMBINE>
__global__ void k_update(Grid g, Box box, const double *__restrict__ Uin, const double *__restrict__ F,
                         double *__restrict__ Uout, const StepParams *__restrict__ P)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    const int slot[5] = { 0, 1, 2, 3, 4 };        // flux slots of rho, mx, my, mz, E
    const int var[5]  = { 0, 1, 2, 3, 7 };
#pragma unroll
    for (int q = 0; q < 5; q++) {
        double u = Uin[var[q] * sa + c];
        for (int d = 0; d < 3; d++) {
            if (!g.act[d]) continue;
            const double *Fd = F + (long long)(d * 8 + slot[q]) * sa + c;
            u -= P->dtdx[d] * (Fd[g.st[d]] - Fd[0]);
        }
        Uout[var[q] * sa + c] = COMBINE ? 0.5 * (Uout[var[q] * sa + c] + u) : u;
    }
    if (!g.act[2]) {
        // 2D: B_z is cell centred and flux updated: F_x[B_z] is x's second induction flux, F_y[B_z] y's first
        double u = Uin[6 * sa + c];
        const double *Fx = F + (long long)(0 * 8 + 6) * sa + c;
        const double *Fy = F + (long long)(1 * 8 + 5) * sa + c;
        u -= P->dtdx[0] * (Fx[g.st[0]] - Fx[0]);
        u -= P->dtdx[1] * (Fy[g.st[1]] - Fy[0]);
        Uout[6 * sa + c] = COMBINE ? 0.5 * (Uout[6 * sa + c] + u) : u;
    }
}

// ---------------------------------------------------------------- CT: edge EMF (a6, R6)
// Component EC of the edge EMF at (a-1/2, b-1/2) of cell c, (EC, a, b) cyclic: arithmetic mean of
// the four face EMFs plus the upwinded half-cell differences to the cell-centred EMFs.
template <int EC>
__global__ void k_emf(Grid g, Box box, const double *__restrict__ V, const double *__restrict__ F,
                      double *__restrict__ Eg)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    constexpr int A = (EC + 1) % 3, B = (EC + 2) % 3;
    const long long c = g.at(i, j, k), sa = g.sa, sA = g.st[A], sB = g.st[B];
    const double *Fa = F + (long long)(A * 8 + 5) * sa;   // F_a[B_b]: first induction flux of sweep a
    const double *Fb = F + (long long)(B * 8 + 6) * sa;   // F_b[B_a]: second induction flux of sweep b
    const double *Wa = F + (long long)(A * 8 + 7) * sa;
    const double *Wb = F + (long long)(B * 8 + 7) * sa;
    const long long c11 = c, c01 = c - sA, c10 = c - sB, c00 = c - sA - sB;
    auto ecell = [&](long long cc) {            // E^c = -(v x B) component EC = v_b B_a - v_a B_b
        return V[(1 + B) * sa + cc] * V[(4 + A) * sa + cc] - V[(1 + A) * sa + cc] * V[(4 + B) * sa + cc];
    };
    double Ea_lo = -Fa[c10], Ea_hi = -Fa[c11];
    double Eb_lo =  Fb[c01], Eb_hi =  Fb[c11];
    double wa_lo = Wa[c10], wa_hi = Wa[c11], wb_lo = Wb[c01], wb_hi = Wb[c11];
    double e00 = ecell(c00), e10 = ecell(c10), e01 = ecell(c01), e11 = ecell(c11);
    double t1 = wa_lo * (Eb_lo - e00) + (1.0 - wa_lo) * (Eb_hi - e10);
    double t2 = wa_hi * (e01 - Eb_lo) + (1.0 - wa_hi) * (e11 - Eb_hi);
    double t3 = wb_lo * (Ea_lo - e00) + (1.0 - wb_lo) * (Ea_hi - e01);
    double t4 = wb_hi * (e10 - Ea_lo) + (1.0 - wb_hi) * (e11 - Ea_hi);
    Eg[EC * sa + c] = 0.25 * (Ea_lo + Ea_hi + Eb_lo + Eb_hi) + 0.25 * (t1 - t2) + 0.25 * (t3 - t4);
}

// ---------------------------------------------------------------- CT: face update  db/dt = -curl E
template <int DIR, bool COMBINE>
__global__ void k_ctface(Grid g, Box box, const double *__restrict__ bin, const double *__restrict__ Eg,
                         double *__restrict__ bout, const StepParams *__restrict__ P)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    const long long c = g.at(i, j, k), sa = g.sa;
    double term1 = 0.0, term2 = 0.0;
    if (g.act[T1]) { const double *E2 = Eg + T2 * sa + c; term1 = (E2[g.st[T1]] - E2[0]) / g.dx[T1]; }
    if (g.act[T2]) { const double *E1 = Eg + T1 * sa + c; term2 = (E1[g.st[T2]] - E1[0]) / g.dx[T2]; }
    double b = bin[DIR * sa + c] - P->dt * (term1 - term2);
    bout[DIR * sa + c] = COMBINE ? 0.5 * (bout[DIR * sa + c] + b) : b;
}

// ---------------------------------------------------------------- cell-centred B := face mean (R7)
__global__ void k_cellb(Grid g, Box box, const double *__restrict__ b, double *__restrict__ U)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    for (int d = 0; d < 3; d++)
        if (g.act[d]) U[(4 + d) * sa + c] = 0.5 * (b[d * sa + c] + b[d * sa + c + g.st[d]]);
}

// ---------------------------------------------------------------- API layout <-> padded layout
// The caller's interior-only array (extent m[] = n[] + face bump) <-> padded array.
__global__ void k_unpack(Grid g, Box box, const double *__restrict__ src, int m0, int m1, double *__restrict__ dst)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    dst[g.at(i, j, k)] = src[((long long)k * m1 + j) * m0 + i];
}

__global__ void k_pack(Grid g, Box box, const double *__restrict__ src, int m0, int m1, double *__restrict__ dst)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    // periodic wrap so the duplicate upper face (index n) and interior-indexed work arrays both come out right
    int ii = i % g.n[0], jj = j % g.n[1], kk = k % g.n[2];
    dst[((long long)k * m1 + j) * m0 + i] = src[g.at(ii, jj, kk)];
}

} // namespace pluto
