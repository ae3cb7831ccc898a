// kernels.cuh -- CUDA kernels of the MHD step (sm_100a).
//
// Per RK stage:   k_ghost<0,1,2>   periodic ghost fill of the 8 cell variables + face fields (a1)
//                 k_sweep_x        cons->prim + PLM + HLLD + flux difference along x (a2-a5), "flat pencil"
//                 k_sweep_march<1> the same along y, each thread marching up its own column
//                 k_sweep_march<2> the same along z
//                 k_emf            CT edge EMFs from the face data the sweeps left (a6)
//                 k_ctface         face-B curl update [+ RK2 combine] (a6, a7)
//                 k_cellb          cell-centred B := face mean
// x is the contiguous index everywhere, so every warp access is a contiguous row segment.
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

__device__ __forceinline__ int wrap_m1(int i, int n) { return i == 0 ? n - 1 : i - 1; }
__device__ __forceinline__ int wrap_p1(int i, int n) { return i == n - 1 ? 0 : i + 1; }

// ---------------------------------------------------------------- periodic ghost fill (a1)
// Fill the ghost layers of `narr` consecutive arrays along AXIS: index g in [-ng,0) <- g + n,
// g in [n, n+ng] <- g - n (cells and faces alike; face n duplicates face 0).  Launched x, then y,
// then z over the full padded extent of the other axes so edges and corners come out right
// (the paper exchanges with diagonal neighbours for the same reason).
__global__ void k_ghost_x(Grid g, double *__restrict__ base)
{
    // one thread per padded row (j,k); the 2*ng+1 ghost cells of a row are strided by nothing
    // useful, so each thread walks them itself
    const long long rows = (long long)g.tot[1] * g.tot[2];
    long long r = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (r >= rows) return;
    double *a = base + (long long)blockIdx.y * g.sa + r * g.st[1] + g.off[0];
    const int n = g.n[0];
    for (int s = 1; s <= g.ng; s++) a[-s] = a[n - s];
    for (int s = 0; s <= g.ng; s++) a[n + s] = a[s];
}

template <int AXIS>   // AXIS = 1 or 2
__global__ void k_ghost_yz(Grid g, double *__restrict__ base, int narr)
{
    const int nghost = 2 * g.ng + 1;
    int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= g.tot[0]) return;
    int slot, other, arr;
    if (AXIS == 1) { slot = blockIdx.y; other = blockIdx.z % g.tot[2]; arr = blockIdx.z / g.tot[2]; }
    else           { other = blockIdx.y; slot = blockIdx.z % nghost;   arr = blockIdx.z / nghost; }
    if (arr >= narr) return;
    const int n = g.n[AXIS];
    int gi = slot < g.ng ? slot - g.ng : n + (slot - g.ng);
    int src = gi < 0 ? gi + n : gi - n;
    double *a = base + (long long)arr * g.sa + x;
    if (AXIS == 1) {
        a += (long long)other * g.st[2];
        a[(long long)(gi + g.off[1]) * g.st[1]] = a[(long long)(src + g.off[1]) * g.st[1]];
    } else {
        a += (long long)other * g.st[1];
        a[(long long)(gi + g.off[2]) * g.st[2]] = a[(long long)(src + g.off[2]) * g.st[2]];
    }
}

// ---------------------------------------------------------------- layout of the CT work arrays
// ct + CT_FEM + 2*d + q : induction flux q of sweep d  (d = x: F_x[By], F_x[Bz]; y: F_y[Bz], F_y[Bx];
//                         z: F_z[Bx], F_z[By]) on the lower d-face of each interior cell
// ct + CT_W + d         : upwind weight on that face
// ct + CT_EC + e        : cell-centred EMF component e, E^c = -(v x B)
// ct + CT_EG + e        : edge EMF component e at the lower (a,b) edge of each interior cell
enum { CT_FEM = 0, CT_W = 6, CT_EC = 9, CT_EG = 12, CT_COUNT = 15 };

// ---------------------------------------------------------------- x sweep (a2-a5 fused)
// The rows of the grid are laid end to end as one list of "items" (cells -2 .. nx+1 of each row).
// A block takes NT consecutive items: every thread loads its cell and converts it to primitives in
// shared memory, limits its own slopes from its two list neighbours, solves the Riemann problem on
// its lower face with its left neighbour's q^L, and differences its flux with its right neighbour's.
// Consecutive blocks overlap by 4 items, so no flux is computed twice inside a block and rows of any
// length pack without a ragged tail.
constexpr int SX_NT = 128;
constexpr int SX_OUT = SX_NT - 4;

template <int LIM, bool TWO_D>
__global__ void __launch_bounds__(SX_NT, 4)
k_sweep_x(Grid g, const double *__restrict__ Uin, const double *__restrict__ bx, double *Uout,
          double *__restrict__ ct, StepParams *P, int combine)
{
    __shared__ double sP[8][SX_NT];     // primitives; rows 0..5 are reused for the fluxes
    __shared__ double sQ[7][SX_NT];     // q^L = q + slope/2 of each cell
    const int t = threadIdx.x;
    const int nx = g.n[0], M = nx + 4;
    const long long sa = g.sa;
    const long long nitems = (long long)M * g.n[1] * g.n[2];
    const long long item = (long long)blockIdx.x * SX_OUT - 2 + t;
    const bool valid = item >= 0 && item < nitems;
    int f = -100;
    long long c = 0;
    double rho = 1.0, mx = 0, my = 0, mz = 0, En = 0, Bzc = 0;
    double q[7] = { 1, 0, 0, 0, 0, 0, 1 };    // rho, vx, vy, vz, By, Bz, p
    double Bxc = 0, bxf = 0;
    double o0 = 0, o1 = 0, o2 = 0, o3 = 0, o6 = 0, o7 = 0;   // S^n of the cell (combine stage)
    if (valid) {
        long long row = item / M;
        f = (int)(item - row * M) - 2;
        int j = (int)(row % g.n[1]), k = (int)(row / g.n[1]);
        c = g.at(f, j, k);
        rho = Uin[c]; mx = Uin[sa + c]; my = Uin[2 * sa + c]; mz = Uin[3 * sa + c];
        Bxc = Uin[4 * sa + c];
        double By = Uin[5 * sa + c];
        Bzc = Uin[6 * sa + c];
        En = Uin[7 * sa + c];
        bxf = bx[c];
        if (combine && f >= 0 && f < nx) {     // issued with the other loads: one memory round trip per block
            o0 = Uout[c]; o1 = Uout[sa + c]; o2 = Uout[2 * sa + c]; o3 = Uout[3 * sa + c]; o7 = Uout[7 * sa + c];
            if (TWO_D) o6 = Uout[6 * sa + c];
        }
        double ir = rcp_fast(rho);
        q[0] = rho; q[1] = mx * ir; q[2] = my * ir; q[3] = mz * ir; q[4] = By; q[5] = Bzc;
        q[6] = (g.gamma - 1.0) * (En - 0.5 * (mx * q[1] + my * q[2] + mz * q[3]) - 0.5 * (Bxc * Bxc + By * By + Bzc * Bzc));
        if (f >= 0 && f < nx && (!(rho > 0.0) || !(q[6] > 0.0) || isinf(rho) || isinf(q[6]))) P->err = 1;
    }
#pragma unroll
    for (int v = 0; v < 7; v++) sP[v][t] = q[v];
    __syncthreads();

    // limited slopes of the own cell (needs both list neighbours, which lie in the same row)
    const bool has_nb = valid && t >= 1 && t <= SX_NT - 2 && f >= -1 && f <= nx;
    double qR[7];
    if (has_nb) {
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double s = plm_slope<LIM>(q[v] - sP[v][t - 1], sP[v][t + 1] - q[v]);
            sQ[v][t] = q[v] + 0.5 * s;
            qR[v] = q[v] - 0.5 * s;
        }
    }
    __syncthreads();

    // Riemann problem on the lower face of cell f (faces 0 .. nx)
    const bool face = has_nb && t >= 2 && f >= 0;
    double F[7] = { 0, 0, 0, 0, 0, 0, 0 }, w = 0.5;
    if (face) {
        Side L = { sQ[0][t - 1], sQ[1][t - 1], sQ[2][t - 1], sQ[3][t - 1], sQ[4][t - 1], sQ[5][t - 1], sQ[6][t - 1] };
        Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
        hlld(L, R, bxf, g.gamma, g.igm1, F, w);
        sP[0][t] = F[0]; sP[1][t] = F[1]; sP[2][t] = F[2]; sP[3][t] = F[3]; sP[4][t] = F[6];
        if (TWO_D) sP[5][t] = F[5];
    }
    __syncthreads();

    // cell f in [0, nx): flux difference with the right neighbour's face, CT data of the own face
    if (face && f < nx && t <= SX_NT - 3) {
        const double dtdx = P->dtdx[0];
        double r0 = rho - dtdx * (sP[0][t + 1] - F[0]);
        double r1 = mx - dtdx * (sP[1][t + 1] - F[1]);
        double r2 = my - dtdx * (sP[2][t + 1] - F[2]);
        double r3 = mz - dtdx * (sP[3][t + 1] - F[3]);
        double r7 = En - dtdx * (sP[4][t + 1] - F[6]);
        if (combine) {
            r0 = 0.5 * (o0 + r0); r1 = 0.5 * (o1 + r1); r2 = 0.5 * (o2 + r2);
            r3 = 0.5 * (o3 + r3); r7 = 0.5 * (o7 + r7);
        }
        Uout[c] = r0; Uout[sa + c] = r1; Uout[2 * sa + c] = r2; Uout[3 * sa + c] = r3; Uout[7 * sa + c] = r7;
        if (TWO_D) {   // B_z has no faces in 2D: cell centred, flux updated
            double r6 = Bzc - dtdx * (sP[5][t + 1] - F[5]);
            Uout[6 * sa + c] = combine ? 0.5 * (o6 + r6) : r6;
        }
        ct[(CT_FEM + 0) * sa + c] = F[4];
        ct[(CT_FEM + 1) * sa + c] = F[5];
        ct[(CT_W + 0) * sa + c] = w;
        // cell-centred EMF  E^c = -(v x B)
        ct[(CT_EC + 0) * sa + c] = q[3] * q[4] - q[2] * q[5];
        ct[(CT_EC + 1) * sa + c] = q[1] * q[5] - q[3] * Bxc;
        ct[(CT_EC + 2) * sa + c] = q[2] * Bxc - q[1] * q[4];
    }
}

// ---------------------------------------------------------------- y / z sweep (a2-a5 fused), marching
// Thread = one column (fixed i and transverse index), marching along DIR over `seglen` cells.  It
// keeps the running q^L, the last two primitive states (as state + difference) and the previous
// flux in registers, so every cell is loaded and converted once and every flux is computed once per
// segment (+1 at the segment end).  Uout already holds the x-sweep result and is updated in place:
//     Uout -= scale * dt/dx_d * (F_d(+) - F_d(-)),  scale = 1 (stage 1) or 1/2 (combine stage).
// cons -> rotated primitives of one cell (Eq. 7)
template <int DIR>
__device__ __forceinline__ void prim_rot(double rho, const double m[3], const double B[3], double En, double gamma,
                                         double q[7], bool &bad)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    double ir = rcp_fast(rho);
    double v[3] = { m[0] * ir, m[1] * ir, m[2] * ir };
    double p = (gamma - 1.0) * (En - 0.5 * (m[0] * v[0] + m[1] * v[1] + m[2] * v[2])
                                   - 0.5 * (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]));
    q[0] = rho; q[1] = v[DIR]; q[2] = v[T1]; q[3] = v[T2]; q[4] = B[T1]; q[5] = B[T2]; q[6] = p;
    bad = !(rho > 0.0) || !(p > 0.0) || isinf(rho) || isinf(p);
}

template <int DIR>
__device__ __forceinline__ void load_rot(const double *__restrict__ U, long long sa, long long c, double gamma,
                                         double q[7], bool &bad)
{
    double m[3] = { U[sa + c], U[2 * sa + c], U[3 * sa + c] };
    double B[3] = { U[4 * sa + c], U[5 * sa + c], U[6 * sa + c] };
    prim_rot<DIR>(U[c], m, B, U[7 * sa + c], gamma, q, bad);
}

// 8-byte asynchronous global -> shared copy (LDGSTS): the data of the next march iteration is in
// flight while the current interface is being solved, at no cost in registers
__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int MARCH_NT = 128;
constexpr int MARCH_PF = 16;     // doubles prefetched per thread and iteration: U(s+1) 8, b_d 1, U'(s-1) 6

template <int DIR, int LIM, bool TWO_D>
__global__ void __launch_bounds__(MARCH_NT, 4)
k_sweep_march(Grid g, const double *__restrict__ Uin, const double *__restrict__ bn, double *Uout,
              double *__restrict__ ct, StepParams *P, double scale, int seglen)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    constexpr bool BZ2D = TWO_D && DIR == 1;           // F_y[B_z] updates the cell-centred B_z in 2D
    __shared__ double pf[2][MARCH_PF][MARCH_NT];
    const int t = threadIdx.x;
    const int i = blockIdx.x * blockDim.x + t;
    if (i >= g.n[0]) return;
    // DIR = 1: grid.y = segment, grid.z = k;   DIR = 2: grid.y = j, grid.z = segment
    const int seg = DIR == 1 ? blockIdx.y : blockIdx.z;
    const int tr = DIR == 1 ? blockIdx.z : blockIdx.y;
    const int s0 = seg * seglen;
    const int s1 = min(s0 + seglen, g.n[DIR]);
    const long long sa = g.sa, st = g.st[DIR];
    long long c = DIR == 1 ? g.at(i, s0, tr) : g.at(i, tr, s0);   // cell s0 of the segment
    const double gamma = g.gamma;
    const double fac = scale * P->dtdx[DIR];
    bool bad, anybad = false;

    // what iteration s consumes: U of cell s+1, the face field on face s-1/2, U' of cell s-1
    auto prefetch = [&](int slot, long long cs) {
#pragma unroll
        for (int v = 0; v < 8; v++) cp_async8(&pf[slot][v][t], Uin + v * sa + cs + st);
        cp_async8(&pf[slot][8][t], bn + cs);
        const long long cm = cs - st;
        cp_async8(&pf[slot][9][t], Uout + cm);
        cp_async8(&pf[slot][10][t], Uout + (1 + DIR) * sa + cm);
        cp_async8(&pf[slot][11][t], Uout + (1 + T1) * sa + cm);
        cp_async8(&pf[slot][12][t], Uout + (1 + T2) * sa + cm);
        cp_async8(&pf[slot][13][t], Uout + 7 * sa + cm);
        if (BZ2D) cp_async8(&pf[slot][14][t], Uout + 6 * sa + cm);
        cp_async_commit();
    };
    prefetch(0, c);

    double qm[7], q0[7], d0[7], qL[7];
    load_rot<DIR>(Uin, sa, c - 2 * st, gamma, qm, bad);
    load_rot<DIR>(Uin, sa, c - st, gamma, q0, bad);
#pragma unroll
    for (int v = 0; v < 7; v++) d0[v] = q0[v] - qm[v];
    load_rot<DIR>(Uin, sa, c, gamma, qm, bad);          // qm now holds cell s0
    anybad |= bad;
#pragma unroll
    for (int v = 0; v < 7; v++) {
        double d1 = qm[v] - q0[v];
        qL[v] = q0[v] + 0.5 * plm_slope<LIM>(d0[v], d1);   // q^L of face s0 - 1/2
        q0[v] = qm[v];
        d0[v] = d1;
    }
    double Fp[6] = { 0, 0, 0, 0, 0, 0 };                // previous face: rho, m_n, m_t1, m_t2, E, (B_z in 2D)

    for (int s = s0; s <= s1; s++, c += st) {
        const int slot = (s - s0) & 1;
        if (s < s1) { prefetch(slot ^ 1, c + st); cp_async_wait<1>(); }
        else        { cp_async_wait<0>(); }
        // cell s is in q0 (with d0 = q_s - q_{s-1}); cell s+1 arrives through shared memory
        double q1[7];
        {
            double m[3], B[3];
            m[0] = pf[slot][1][t]; m[1] = pf[slot][2][t]; m[2] = pf[slot][3][t];
            B[0] = pf[slot][4][t]; B[1] = pf[slot][5][t]; B[2] = pf[slot][6][t];
            prim_rot<DIR>(pf[slot][0][t], m, B, pf[slot][7][t], gamma, q1, bad);
        }
        if (s + 1 < s1) anybad |= bad;
        double qR[7];
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double d1 = q1[v] - q0[v];
            double sl = plm_slope<LIM>(d0[v], d1);
            qR[v] = q0[v] - 0.5 * sl;
            double nl = q0[v] + 0.5 * sl;
            q0[v] = q1[v];
            d0[v] = d1;
            q1[v] = nl;                                   // q1 now carries the next q^L
        }
        Side L = { qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6] };
        Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
        double F[7], w;
        hlld(L, R, pf[slot][8][t], gamma, g.igm1, F, w);
#pragma unroll
        for (int v = 0; v < 7; v++) qL[v] = q1[v];
        if (s > s0) {
            const long long cm = c - st;                  // cell s-1
            Uout[cm] = pf[slot][9][t] - fac * (F[0] - Fp[0]);
            Uout[(1 + DIR) * sa + cm] = pf[slot][10][t] - fac * (F[1] - Fp[1]);
            Uout[(1 + T1) * sa + cm] = pf[slot][11][t] - fac * (F[2] - Fp[2]);
            Uout[(1 + T2) * sa + cm] = pf[slot][12][t] - fac * (F[3] - Fp[3]);
            Uout[7 * sa + cm] = pf[slot][13][t] - fac * (F[6] - Fp[4]);
            if (BZ2D) Uout[6 * sa + cm] = pf[slot][14][t] - fac * (F[4] - Fp[5]);   // F_y[B_z]
        }
        if (s < s1) {
            ct[(CT_FEM + 2 * DIR) * sa + c] = F[4];
            ct[(CT_FEM + 2 * DIR + 1) * sa + c] = F[5];
            ct[(CT_W + DIR) * sa + c] = w;
        }
        Fp[0] = F[0]; Fp[1] = F[1]; Fp[2] = F[2]; Fp[3] = F[3]; Fp[4] = F[6]; Fp[5] = F[4];
    }
    if (anybad) P->err = 1;
}

// ---------------------------------------------------------------- CT: edge EMFs (a6, R6)
// Thread = interior cell; computes the EMF components on its three lower edges (only E_z in 2D):
// arithmetic mean of the four face EMFs plus the upwinded half-cell differences to the cell-centred
// EMFs.  Neighbours are taken with periodic wrap, so the CT work arrays need no ghost layers.
template <int EC>
__device__ __forceinline__ double edge_emf(const Grid &g, const double *__restrict__ ct, int i, int j, int k)
{
    constexpr int A = (EC + 1) % 3, B = (EC + 2) % 3;
    const long long sa = g.sa;
    int p[3] = { i, j, k };
    int pa[3] = { i, j, k }, pb[3] = { i, j, k }, pab[3] = { i, j, k };
    pa[A] = wrap_m1(p[A], g.n[A]);
    pb[B] = wrap_m1(p[B], g.n[B]);
    pab[A] = pa[A]; pab[B] = pb[B];
    const long long c11 = g.at(p[0], p[1], p[2]), c01 = g.at(pa[0], pa[1], pa[2]);
    const long long c10 = g.at(pb[0], pb[1], pb[2]), c00 = g.at(pab[0], pab[1], pab[2]);
    const double *Fa = ct + (CT_FEM + 2 * A) * sa;       // F_a[B_b]: first induction flux of sweep a
    const double *Fb = ct + (CT_FEM + 2 * B + 1) * sa;   // F_b[B_a]: second induction flux of sweep b
    const double *Wa = ct + (CT_W + A) * sa, *Wb = ct + (CT_W + B) * sa;
    const double *Ec = ct + (CT_EC + EC) * sa;
    double Ea_lo = -Fa[c10], Ea_hi = -Fa[c11];
    double Eb_lo =  Fb[c01], Eb_hi =  Fb[c11];
    double wa_lo = Wa[c10], wa_hi = Wa[c11], wb_lo = Wb[c01], wb_hi = Wb[c11];
    double e00 = Ec[c00], e10 = Ec[c10], e01 = Ec[c01], e11 = Ec[c11];
    double t1 = wa_lo * (Eb_lo - e00) + (1.0 - wa_lo) * (Eb_hi - e10);
    double t2 = wa_hi * (e01 - Eb_lo) + (1.0 - wa_hi) * (e11 - Eb_hi);
    double t3 = wb_lo * (Ea_lo - e00) + (1.0 - wb_lo) * (Ea_hi - e01);
    double t4 = wb_hi * (e10 - Ea_lo) + (1.0 - wb_hi) * (e11 - Ea_hi);
    return 0.25 * (Ea_lo + Ea_hi + Eb_lo + Eb_hi) + 0.25 * (t1 - t2) + 0.25 * (t3 - t4);
}

__global__ void k_emf(Grid g, Box box, double *__restrict__ ct)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    double ez = edge_emf<2>(g, ct, i, j, k);
    if (g.act[2]) {
        double ex = edge_emf<0>(g, ct, i, j, k);
        double ey = edge_emf<1>(g, ct, i, j, k);
        ct[(CT_EG + 0) * sa + c] = ex;
        ct[(CT_EG + 1) * sa + c] = ey;
    }
    ct[(CT_EG + 2) * sa + c] = ez;
}

// ---------------------------------------------------------------- CT: face update  db/dt = -curl E  [+ combine (a7)]
// Thread = interior cell, updates its three lower faces; the +1 edge neighbours wrap periodically.
// COMBINE: bout <- (bout + that)/2 in place (bout holds the faces of S^n).
template <bool COMBINE>
__global__ void k_ctface(Grid g, Box box, const double *__restrict__ bin, const double *__restrict__ ct,
                         double *bout, const StepParams *__restrict__ P)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    const double dt = P->dt;
    const double *Ex = ct + (CT_EG + 0) * sa, *Ey = ct + (CT_EG + 1) * sa, *Ez = ct + (CT_EG + 2) * sa;
    const long long cxp = g.at(wrap_p1(i, g.n[0]), j, k);
    const long long cyp = g.at(i, wrap_p1(j, g.n[1]), k);
    const double ez = Ez[c];
    double bxn, byn;
    if (g.act[2]) {
        const long long czp = g.at(i, j, wrap_p1(k, g.n[2]));
        const double ex = Ex[c], ey = Ey[c];
        bxn = bin[c] - dt * ((Ez[cyp] - ez) / g.dx[1] - (Ey[czp] - ey) / g.dx[2]);
        byn = bin[sa + c] - dt * ((Ex[czp] - ex) / g.dx[2] - (Ez[cxp] - ez) / g.dx[0]);
        double bzn = bin[2 * sa + c] - dt * ((Ey[cxp] - ey) / g.dx[0] - (Ex[cyp] - ex) / g.dx[1]);
        bout[2 * sa + c] = COMBINE ? 0.5 * (bout[2 * sa + c] + bzn) : bzn;
    } else {
        bxn = bin[c] - dt * ((Ez[cyp] - ez) / g.dx[1] - 0.0);
        byn = bin[sa + c] - dt * (0.0 - (Ez[cxp] - ez) / g.dx[0]);
    }
    bout[c] = COMBINE ? 0.5 * (bout[c] + bxn) : bxn;
    bout[sa + c] = COMBINE ? 0.5 * (bout[sa + c] + byn) : byn;
}

// ---------------------------------------------------------------- cell-centred B := face mean (R7)
__global__ void k_cellb(Grid g, Box box, const double *__restrict__ b, double *__restrict__ U)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    U[4 * sa + c] = 0.5 * (b[c] + b[g.at(wrap_p1(i, g.n[0]), j, k)]);
    U[5 * sa + c] = 0.5 * (b[sa + c] + b[sa + g.at(i, wrap_p1(j, g.n[1]), k)]);
    if (g.act[2]) U[6 * sa + c] = 0.5 * (b[2 * sa + c] + b[2 * sa + g.at(i, j, wrap_p1(k, g.n[2]))]);
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
    // periodic wrap: the duplicate upper face (index n) is face 0
    int ii = i % g.n[0], jj = j % g.n[1], kk = k % g.n[2];
    dst[((long long)k * m1 + j) * m0 + i] = src[g.at(ii, jj, kk)];
}

} // namespace pluto
