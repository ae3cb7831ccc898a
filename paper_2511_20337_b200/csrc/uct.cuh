// uct.cuh -- constrained transport with the UCT-HLLD EMF average ([47] named at PAPER.md:271, reference entry
// :640; reading R19 in DESIGN.md).  The sweeps (fused x+y with PLM, one kernel per direction with WENO-Z) call
// hlld_t<true>, which leaves a^L, d^L, d^R and the two transverse velocities on every face; then
//   k_uct_halo   periodic x / y halos of the 15 face arrays (the reconstruction along a transverse direction
//                reaches 2 cells with PLM, 3 with WENO-Z),
//   k_emf_uct    the three edge EMFs, one thread per edge triple, into three work arrays,
//   k_ct_update  face update  db/dt = -curl E  [+ Runge-Kutta combine].
#pragma once
#include "kernels.cuh"

namespace pluto {

// the 15 face arrays [direction d][a^L, d^L, d^R, vbar_t1, vbar_t2] and the edge EMFs E_x, E_y, E_z
struct UctArrays { double *p[UCT_COUNT]; };

// Every halo position (i or j outside the interior, within h) of the 15 face arrays receives its periodic image;
// sources are interior positions, so there is no ordering between copies.  grid.x = chunk of UCT_HALO_ROWS padded
// rows (j = -h .. n1 + h - 1), grid.y = plane (k = -hz .. n2 + hz - 1), grid.z = array.  Halo rows are copied whole,
// interior rows contribute their 2h end positions (walked as one flat list so that no thread idles).
constexpr int UCT_HALO_ROWS = 32;
__global__ void __launch_bounds__(256) k_uct_halo(Grid g, UctArrays A, int h, int hz)
{
    const int n0 = g.n[0], n1 = g.n[1];
    const int j0 = (int)blockIdx.x * UCT_HALO_ROWS - h, j1 = min(j0 + UCT_HALO_ROWS, n1 + h);
    const int k = (int)blockIdx.y - hz;
    double *arr = A.p[blockIdx.z];
    // whole halo rows of this chunk
    for (int j = j0; j < j1; j++) {
        if (j >= 0 && j < n1) continue;
        const int sj = ((j % n1) + n1) % n1;
        double *dst = arr + g.at(-h, j, k);
        const double *src = arr + g.at(0, sj, k);
        for (int e = threadIdx.x; e < n0 + 2 * h; e += blockDim.x) {
            const int i = e - h;
            dst[e] = src[((i % n0) + n0) % n0];
        }
    }
    // x ends of the interior rows of this chunk
    const int i0 = max(j0, 0), i1 = min(j1, n1);
    for (int t = threadIdx.x; t < (i1 - i0) * 2 * h; t += blockDim.x) {
        const int j = i0 + t / (2 * h), e = t % (2 * h);
        const int i = e < h ? e - h : n0 + (e - h);
        arr[g.at(i, j, k)] = arr[g.at(((i % n0) + n0) % n0, j, k)];
    }
}

// values at the edge between positions -1 and 0 of a quantity on a line with stride st (q points at position 0):
// from below (upper-face value of cell -1) and from above (lower-face value of cell 0), with the reconstruction of the run
template <int LIM>
__device__ __forceinline__ void edge_values(const double *__restrict__ q, long long st, double &below, double &above)
{
    const double m2 = q[-2 * st], m1 = q[-st], p0 = q[0], p1 = q[st];
    if (LIM == 2) {
        const double m3 = q[-3 * st], p2 = q[2 * st];
        below = wenoz_upper(m3, m2, m1, p0, p1);
        above = wenoz_upper(p2, p1, p0, m1, m2);
    } else {
        double lo, hi;
        plm_faces<LIM == 2 ? 0 : LIM>(m1, m1 - m2, p0 - m1, lo, below);
        plm_faces<LIM == 2 ? 0 : LIM>(p0, p0 - m1, p1 - p0, above, hi);
    }
}

// E_e = v_b B_a - v_a B_b at the edge (a - 1/2, b - 1/2) of cell c, (e, a, b) cyclic (reading R19):
//   E_e = -[a_a^W (vbar_a B_b)^W + a_a^E (vbar_a B_b)^E] + [a_b^S (vbar_b B_a)^S + a_b^N (vbar_b B_a)^N]
//         + (d_a^E B_b^E - d_a^W B_b^W) - (d_b^N B_a^N - d_b^S B_a^S)
// W / E: below / above the edge along a, S / N: below / above it along b.  B_b, vbar_a: the staggered field and the
// transverse velocity on the two b-faces meeting at the edge, reconstructed along a up to the edge; B_a, vbar_b:
// likewise on the two a-faces along b.  a_a, d_a: coefficients of the two a-interfaces meeting at the edge,
// arithmetic mean of the two; likewise a_b, d_b.
template <int LIM>
__device__ __forceinline__ double uct_edge(const UctArrays &A, const double *__restrict__ bfaces, long long sa,
                                           long long c, int a, int b, long long sta, long long stb)
{
    // a-interfaces below (c - stb) and above (c) the edge along b; b-interfaces below (c - sta) / above (c) along a
    const double *aLa = A.p[a * 5 + 0], *dLa = A.p[a * 5 + 1], *dRa = A.p[a * 5 + 2];
    const double *aLb = A.p[b * 5 + 0], *dLb = A.p[b * 5 + 1], *dRb = A.p[b * 5 + 2];
    const double aW = 0.5 * (aLa[c - stb] + aLa[c]), aE = 0.5 * ((1.0 - aLa[c - stb]) + (1.0 - aLa[c]));
    const double dW = 0.5 * (dLa[c - stb] + dLa[c]), dE = 0.5 * (dRa[c - stb] + dRa[c]);
    const double aS = 0.5 * (aLb[c - sta] + aLb[c]), aN = 0.5 * ((1.0 - aLb[c - sta]) + (1.0 - aLb[c]));
    const double dS = 0.5 * (dLb[c - sta] + dLb[c]), dN = 0.5 * (dRb[c - sta] + dRb[c]);
    // on b-faces vbar_a is the second transverse velocity of direction b; on a-faces vbar_b is the first of direction a
    double BbW, BbE, vaW, vaE, BaS, BaN, vbS, vbN;
    edge_values<LIM>(bfaces + b * sa + c, sta, BbW, BbE);
    edge_values<LIM>(A.p[b * 5 + 4] + c, sta, vaW, vaE);
    edge_values<LIM>(bfaces + a * sa + c, stb, BaS, BaN);
    edge_values<LIM>(A.p[a * 5 + 3] + c, stb, vbS, vbN);
    return -fma(aW * vaW, BbW, aE * vaE * BbE) + fma(aS * vbS, BaS, aN * vbN * BaN)
           + fma(dE, BbE, -dW * BbW) - fma(dN, BaN, -dS * BaS);
}

// one thread per cell (i, j, k) of [0, n0] x [0, n1] x [0, n2]: the EMFs on its three lower edges.  Blocks are
// UCT_TX x UCT_TY tiles of one plane: the stencils of neighbouring rows meet in L1.
constexpr int UCT_TX = 32, UCT_TY = 4;
template <int LIM, bool TWO_D>
__global__ void __launch_bounds__(UCT_TX * UCT_TY) k_emf_uct(Grid g, UctArrays A, const double *__restrict__ bfaces)
{
    const int i = blockIdx.x * UCT_TX + threadIdx.x, j = blockIdx.y * UCT_TY + threadIdx.y, k = blockIdx.z;
    if (i > g.n[0] || j > g.n[1]) return;
    const long long c = g.at(i, j, k), sa = g.sa;
    A.p[UCT_FACE + 2][c] = uct_edge<LIM>(A, bfaces, sa, c, 0, 1, 1, g.st[1]);                 // E_z: a = x, b = y
    if (!TWO_D) {
        A.p[UCT_FACE + 0][c] = uct_edge<LIM>(A, bfaces, sa, c, 1, 2, g.st[1], g.st[2]);       // E_x: a = y, b = z
        A.p[UCT_FACE + 1][c] = uct_edge<LIM>(A, bfaces, sa, c, 2, 0, g.st[2], 1);             // E_y: a = z, b = x
    }
}

// one thread per cell (i, j, k) of [0, n0) x [0, n1) x [0, n2] (3D: plane n2 only receives b_z on face n2, kept in
// the ghost plane like k_ct_tma does): b <- b - dt curl E, COMBINE: wn * S^n + ws * that (cb.Sn = the faces of S^n)
template <bool COMBINE, bool TWO_D>
__global__ void __launch_bounds__(128) k_ct_update(Grid g, UctArrays A, const double *__restrict__ bin, double *bout,
                                                   const StepParams *__restrict__ P, Combine cb)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
    if (i >= g.n[0]) return;
    const long long c = g.at(i, j, k), sa = g.sa, st1 = g.st[1], st2 = g.st[2];
    const double dtdx = P->dtdx[0], dtdy = P->dtdx[1], dtdz = P->dtdx[2];
    const double *Ex = A.p[UCT_FACE + 0], *Ey = A.p[UCT_FACE + 1], *Ez = A.p[UCT_FACE + 2];
    auto put = [&](int f, long long at, double v) {
        bout[f * sa + at] = COMBINE ? fma(cb.wn, cb.Sn[f * sa + at], cb.ws * v) : v;
    };
    if (TWO_D || k < g.n[2]) {
        const double ez = Ez[c];
        double bxn = fma(-dtdy, Ez[c + st1] - ez, bin[c]);
        double byn = fma(dtdx, Ez[c + 1] - ez, bin[sa + c]);
        if (!TWO_D) {
            bxn = fma(dtdz, Ey[c + st2] - Ey[c], bxn);
            byn = fma(-dtdz, Ex[c + st2] - Ex[c], byn);
        }
        put(0, c, bxn);
        if (i == 0) bout[c + g.n[0]] = bout[c];      // periodic copy: x-face n0 is face 0 (same thread wrote it)
        put(1, c, byn);
    }
    if (!TWO_D) {
        const double bzn = fma(-dtdx, Ey[c + 1] - Ey[c], fma(dtdy, Ex[c + st1] - Ex[c], bin[2 * sa + c]));
        put(2, c, bzn);
    }
}

} // namespace pluto
