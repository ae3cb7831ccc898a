// kernels.cuh -- CUDA kernels of the MHD step (sm_100a).
//
// Per RK stage:   k_ghost          periodic ghost fill of the 8 state arrays, one launch (a1)
//                 k_sweep_x        cons->prim + PLM + HLLD + flux difference along x (a2-a5), "flat pencil"
//                 k_sweep_march<1> the same along y, each thread marching up its own column
//                 k_sweep_march<2> the same along z
//                 k_ct             CT: edge EMFs from the face data the sweeps left, face-B curl update
//                                  [+ RK2 combine], marching along z with the edge EMFs in shared memory (a6, a7)
// x is the contiguous index everywhere, so every warp access is a contiguous row segment.
// A state is S[0..4] = rho, m_x, m_y, m_z, E and S[5..7] = b_x, b_y, b_z face fields (grid.h).
#pragma once
#include "grid.h"
#include "mhd_device.cuh"

namespace pluto {

struct Box { int lo[3], hi[3]; };   // inclusive lo, exclusive hi

// Runge-Kutta stage combine (a7): the stage writes  wn * S^n + ws * (S + L(S)).  Sn == nullptr: the plain
// Euler stage S + L(S).  SSP-RK2 (R3): (1/2, 1/2).  SSP-RK3 (Eq. 5): (3/4, 1/4), (1/3, 2/3).
// Sn may be the array the stage writes (each value is read before it is overwritten by the same thread).
struct Combine { const double *Sn; double wn, ws; };

__device__ __forceinline__ bool thread_zone(const Box &b, int &i, int &j, int &k)
{
    i = b.lo[0] + blockIdx.x * blockDim.x + threadIdx.x;
    j = b.lo[1] + blockIdx.y;
    k = b.lo[2] + blockIdx.z;
    return i < b.hi[0];
}

__device__ __forceinline__ int wrap_m1(int i, int n) { return i == 0 ? n - 1 : i - 1; }
__device__ __forceinline__ int wrap_p1(int i, int n) { return i == n - 1 ? 0 : i + 1; }

// ---------------------------------------------------------------- mbarrier / TMA primitives (PTX)
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity)
{
    const unsigned a = smem_u32(bar);
    unsigned ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// generic-proxy accesses to shared memory before this point are ordered before later async-proxy (TMA) writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// contiguous bytes global -> shared by the TMA engine (no tensor map; 16-byte aligned, size % 16 == 0),
// completion counted in bytes on `bar`
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, unsigned bytes, void *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------- ghost fill (a1)
// Where the z-ghost planes of a state come from.  A periodic single domain is its own neighbour on
// both sides (lo = hi = the state itself).  In a z-slab decomposition (Fig. 4) lo / hi
// are the same state of the slab below / above -- in this process or, peer-mapped, on another GPU: the
// ghost kernel PULLS the planes it needs straight out of the neighbour's interior (no pack / unpack
// buffers).  x and y stay periodic inside every slab.  All slabs share nx, ny and the ghost count, so
// the in-plane strides agree; the plane count and the array stride may differ.
struct ZSrc {
    const double *lo, *hi;      // array 0 of the neighbour states
    long long lo_sa, hi_sa;     // elements per array there
    int lo_n2, hi_n2;           // interior planes there
};

// source of z-ghost plane k (k < 0 or k >= n2) of array a: pointer to the start of the neighbour's
// array and the interior plane index there (modular: a domain thinner than the ghost depth wraps twice)
__device__ __forceinline__ const double *zsrc_plane(const Grid &g, const ZSrc &z, int a, int k, int &sk)
{
    if (k < 0) { sk = ((k % z.lo_n2) + z.lo_n2) % z.lo_n2; return z.lo + (long long)a * z.lo_sa; }
    sk = (k - g.n[2]) % z.hi_n2;
    return z.hi + (long long)a * z.hi_sa;
}

// Every ghost position (index g in [-ng, 0) or [n, n+ng] along at least one active axis; cells and
// faces alike, face n duplicates face 0) receives the value of its periodic image in the interior:
// index g -> g + n or g - n along every axis at once (along z: the image lies in the neighbour slab).
// Edges and corners therefore come out right in ONE launch (the paper exchanges with diagonal
// neighbours for the same reason), and sources are never written, so there is no
// ordering between positions.  The ghost set is walked as three slab families: z-ghost planes (full
// padded rows), y-ghost rows of interior planes, x-ghost ends of interior rows.
__global__ void __launch_bounds__(256) k_ghost(Grid g, double *__restrict__ base, int narr, ZSrc zs)
{
    const int ng = g.ng, ngh = 2 * ng + 1;
    const int gi = g.n[0] + ngh;                          // x positions -ng .. n+ng
    const int gj = g.act[1] ? g.n[1] + ngh : 1;
    const long long nZ = g.act[2] ? (long long)ngh * gj * gi : 0;
    const long long nY = g.act[1] ? (long long)g.n[2] * ngh * gi : 0;
    const long long nX = (long long)g.n[2] * g.n[1] * ngh;
    const long long total = nZ + nY + nX;
    for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        int i, j, k;
        if (t < nZ) {
            i = (int)(t % gi) - ng;
            long long r = t / gi;
            j = (int)(r % gj) - (g.act[1] ? ng : 0);
            int s = (int)(r / gj);
            k = s < ng ? s - ng : g.n[2] + (s - ng);
        } else if (t < nZ + nY) {
            long long u = t - nZ;
            i = (int)(u % gi) - ng;
            long long r = u / gi;
            int s = (int)(r % ngh);
            j = s < ng ? s - ng : g.n[1] + (s - ng);
            k = (int)(r / ngh);
        } else {
            long long u = t - nZ - nY;
            int s = (int)(u % ngh);
            i = s < ng ? s - ng : g.n[0] + (s - ng);
            long long r = u / ngh;
            j = (int)(r % g.n[1]);
            k = (int)(r / g.n[1]);
        }
        // (extents may be as small as ng, so index n+ng can need two periods)
        const int si = (i + 2 * g.n[0]) % g.n[0], sj = (j + 2 * g.n[1]) % g.n[1];
        const long long dst = g.at(i, j, k);
        if (t < nZ) {
            int sk;
#pragma unroll 8
            for (int a = 0; a < narr; a++) {
                const double *src = zsrc_plane(g, zs, a, k, sk);
                base[a * g.sa + dst] = src[g.at(si, sj, sk)];
            }
        } else {
            const long long src = g.at(si, sj, k);
#pragma unroll 8
            for (int a = 0; a < narr; a++) base[a * g.sa + dst] = base[a * g.sa + src];
        }
    }
}

// Ghost rows and planes only (y and z slabs), as whole padded rows: used when no kernel reads an x ghost
// except the x-face n0, which the CT kernel writes together with face 0.  grid.x = ghost row, grid.y =
// array.  The rows are walked as: the ghost planes (every padded row j of planes -ng..-1, n2..n2+ng), then
// the ghost rows of the interior planes.  A row is copied over the padded x range [-ng, n0+ng].
__global__ void __launch_bounds__(128) k_ghost_yz(Grid g, double *__restrict__ base, ZSrc zs)
{
    const int ng = g.ng, ngh = 2 * ng + 1;
    const int rows_z = g.act[2] ? ngh * (g.n[1] + ngh) : 0;
    int r = blockIdx.x, j, k;
    double *arr = base + (long long)blockIdx.y * g.sa;
    const double *srcarr = arr;
    int sk;
    if (r < rows_z) {
        const int pz = r / (g.n[1] + ngh);
        j = r - pz * (g.n[1] + ngh) - ng;
        k = pz < ng ? pz - ng : g.n[2] + (pz - ng);
        srcarr = zsrc_plane(g, zs, blockIdx.y, k, sk);
    } else {
        r -= rows_z;
        k = r / ngh;
        const int py = r - k * ngh;
        j = py < ng ? py - ng : g.n[1] + (py - ng);
        sk = k;
    }
    const int sj = (j + 2 * g.n[1]) % g.n[1];
    double *dst = arr + g.at(-ng, j, k);
    const double *src = srcarr + g.at(-ng, sj, sk);
    for (int e = threadIdx.x; e < g.n[0] + ngh; e += blockDim.x) dst[e] = src[e];
}

// ---------------------------------------------------------------- layout of the CT work arrays
// ct + CT_FEM + 2*d + q : induction flux q of sweep d  (d = x: F_x[By], F_x[Bz]; y: F_y[Bz], F_y[Bx];
//                         z: F_z[Bx], F_z[By]) on the lower d-face of each interior cell
// ct + CT_W + d         : upwind weight on that face
// ct + CT_EC + e        : cell-centred EMF component e, E^c = -(v x B)
enum { CT_FEM = 0, CT_W = 6, CT_EC = 9, CT_COUNT = 12 };

// UCT-HLLD mode (reading R19): instead of the two induction fluxes and the weight, a sweep along d leaves on the
// lower d-face of every cell the five numbers of hlld_t<true>: a^L, d^L, d^R and the two transverse velocities
// (t1, t2) = (d+1, d+2).  No periodic x copies: k_uct_halo fills the halos of these arrays.
struct UctOut { double *p[5]; };
constexpr int UCT_FACE = 15, UCT_COUNT = 18;      // 3 x 5 face arrays, then the three edge EMFs

// The CT kernel reads the CT arrays one position beyond the interior in x (i = -1 and i = nx hold the
// periodic copies of cells nx-1 and 0).  The sweep kernels write those copies with the value itself:
// offset of the copy for cell i, or 0.
__device__ __forceinline__ int ct_xdup(int i, int nx) { return i == 0 ? nx : (i == nx - 1 ? -nx : 0); }

// cell-centred B of cell c from the face arrays b = S + S_B*sa (R7); 2D: b[2] is the cell-centred B_z
template <bool TWO_D>
__device__ __forceinline__ void cell_b(const Grid &g, const double *__restrict__ b, long long c, double B[3])
{
    B[0] = 0.5 * (b[c] + b[c + 1]);
    B[1] = 0.5 * (b[g.sa + c] + b[g.sa + c + g.st[1]]);
    B[2] = TWO_D ? b[2 * g.sa + c] : 0.5 * (b[2 * g.sa + c] + b[2 * g.sa + c + g.st[2]]);
}

// ---------------------------------------------------------------- CFL pre-filter written by the last stage (a8)
// In 3D the z sweep, which writes the final hydro variables of a step, also leaves, per cell of a coarse
// "bound grid" (grid.h BoundGrid; one cell = the zones one thread finishes: a row of a z segment), an UPPER BOUND of
// every CFL candidate (|v_d| + c_f,d)/dx_d of the zones in it.  The exact reduction of the next step
// (dt_kernel.cu) then only visits rows whose bound can still hold the maximum; the dt stays bit-exact
// because a skipped row provably cannot raise it.  The bound needs no magnetic field (the final faces are
// written later by the CT kernel) and no division per zone:
//     c_f,d^2 <= (gamma p + B^2)/rho,   p >= 0  =>  B^2 <= 2 (E - K) <= 2 E,
//     gamma p + B^2 <= max(gamma (gamma - 1), 2) E   (linear in B^2 on [0, 2E]),
// so with the minimum density, the maximum energy and the maximum of |m_d|/dx_d over the thread's zones
//     (|v_d| + c_f,d)/dx_d <= ( max|m_d|/dx_d + sqrt(cfac E_max rho_min) max(1/dx_d) ) / rho_min.
// The three running values live in shared memory (slot[0], slot[stride], slot[2 stride] of the thread):
// the marching kernels have no registers to spare.
struct SigmaBound {
    double *slot;
    int stride;
    __device__ __forceinline__ void init(double *p, int st) { slot = p; stride = st; p[0] = 1e300; p[st] = 0.0; p[2 * st] = 0.0; }
    __device__ __forceinline__ void add(const Grid &g, double rho, double mx, double my, double mz, double En)
    {
        slot[0] = fmin(slot[0], rho);
        slot[stride] = fmax(slot[stride], En);
        double m = fabs(mx) * g.idx[0];
        if (g.act[1]) m = fmax(m, fabs(my) * g.idx[1]);
        if (g.act[2]) m = fmax(m, fabs(mz) * g.idx[2]);
        slot[2 * stride] = fmax(slot[2 * stride], m);
    }
    // (a NaN never enters fmin / fmax; such a zone is reported by the sweeps' own check)
    __device__ __forceinline__ double value(const Grid &g, double cfac) const
    {
        const double rho_min = slot[0], e_max = slot[stride], m_max = slot[2 * stride];
        double imax = g.idx[0];
        if (g.act[1]) imax = fmax(imax, g.idx[1]);
        if (g.act[2]) imax = fmax(imax, g.idx[2]);
        const double b = (m_max + sqrt(cfac * e_max * rho_min) * imax) / rho_min * (1.0 + 1e-9);
        return (rho_min > 0.0 && b >= 0.0 && b < 1e300) ? b : 1e300;          // unknown: visit the row
    }
};

__device__ __forceinline__ void bound_publish(const BoundGrid &bg, int j, int k, double b)
{
    atomicMax(bg.b + (long long)(k / bg.bk) * bg.nbj + j / bg.bj, (unsigned long long)__double_as_longlong(b));
}

// ---------------------------------------------------------------- x sweep (a2-a5 fused)
// The rows of the grid are laid end to end as one list of "items" (cells -2 .. nx+1 of each row).
// A block takes NT consecutive items: every thread loads its cell and converts it to primitives in
// shared memory, limits its own slopes from its two list neighbours, solves the Riemann problem on
// its lower face with its left neighbour's q^L, and differences its flux with its right neighbour's.
// Consecutive blocks overlap by 4 items, so no flux is computed twice inside a block and rows of any
// length pack without a ragged tail.  The halo cells of a row are its own periodic images.
constexpr int SX_NT = 128;
// halo cells on each side of a block's output range: 2 for PLM, 3 for the five-cell WENO-Z stencil
__host__ __device__ constexpr int sx_halo(int lim) { return lim == 2 ? 3 : 2; }
__host__ __device__ constexpr int sx_out(int lim) { return SX_NT - 2 * sx_halo(lim); }

// hz: planes beyond the interior on each side of a 3D slab whose face data the CT step reads (1; UCT-HLLD: the
// reach of the reconstruction).  UCT: leave the UCT-HLLD face data in uo instead of the CT arrays.
template <int LIM, bool TWO_D, bool UCT>
__global__ void __launch_bounds__(SX_NT, 4)
k_sweep_x(Grid g, const double *__restrict__ Sin, double *Sout, double *__restrict__ ct, StepParams *P, Combine cb,
          int hz, UctOut uo)
{
    __shared__ double sP[8][SX_NT];     // primitives; rows 0..5 are reused for the fluxes
    __shared__ double sQ[7][SX_NT];     // q^L = q + slope/2 of each cell
    const int t = threadIdx.x;
    constexpr int H = sx_halo(LIM);
    const int nx = g.n[0], M = nx + 2 * H;
    const long long sa = g.sa;
    // 3D: planes -hz .. nz + hz - 1 -- the CT kernel reads the x-face data beyond the interior (no z wrap)
    const int nzp = TWO_D ? 1 : g.n[2] + 2 * hz, kz0 = TWO_D ? 0 : -hz;
    const long long nitems = (long long)M * g.n[1] * nzp;
    const long long item = (long long)blockIdx.x * sx_out(LIM) - H + t;
    const bool valid = item >= 0 && item < nitems;
    int f = -100;
    long long c = 0;
    double rho = 1.0, mx = 0, my = 0, mz = 0, En = 0;
    double q[7] = { 1, 0, 0, 0, 0, 0, 1 };    // rho, vx, vy, vz, By, Bz, p
    double Bc[3] = { 0, 0, 0 }, bxf = 0;
    double o0 = 0, o1 = 0, o2 = 0, o3 = 0, o4 = 0, o7 = 0;   // S^n of the cell (combine stage)
    if (valid) {
        long long row = item / M;
        f = (int)(item - row * M) - H;
        int j = (int)(row % g.n[1]), k = (int)(row / g.n[1]) + kz0;
        // halo cells are read from their periodic image (x-face nx is kept equal to face 0 by the CT kernel):
        // no kernel of this path reads an x ghost of the state
        c = g.at(((f % nx) + nx) % nx, j, k);
        rho = Sin[c]; mx = Sin[sa + c]; my = Sin[2 * sa + c]; mz = Sin[3 * sa + c];
        En = Sin[4 * sa + c];
        bxf = Sin[S_B * sa + c];
        cell_b<TWO_D>(g, Sin + S_B * sa, c, Bc);
        if (cb.Sn && f >= 0 && f < nx) {       // issued with the other loads: one memory round trip per block
            const double *Sn = cb.Sn;
            o0 = Sn[c]; o1 = Sn[sa + c]; o2 = Sn[2 * sa + c]; o3 = Sn[3 * sa + c]; o4 = Sn[4 * sa + c];
            if (TWO_D) o7 = Sn[7 * sa + c];
        }
        double ir = rcp_fast(rho);
        q[0] = rho; q[1] = __dmul_rn(mx, ir); q[2] = __dmul_rn(my, ir); q[3] = __dmul_rn(mz, ir);      // see prim_rot
        q[4] = Bc[1]; q[5] = Bc[2];
        q[6] = __dmul_rn(g.gamma - 1.0, fma(-0.5, fma(Bc[0], Bc[0], fma(Bc[1], Bc[1], Bc[2] * Bc[2])),
                                            fma(-0.5, fma(mx, q[1], fma(my, q[2], mz * q[3])), En)));
        if (f >= 0 && f < nx && (unphysical(rho) || unphysical(q[6]))) P->err = 1;
    }
#pragma unroll
    for (int v = 0; v < 7; v++) sP[v][t] = q[v];
    __syncthreads();

    // limited slopes of the own cell (needs both list neighbours, which lie in the same row)
    const bool has_nb = valid && t >= H - 1 && t <= SX_NT - H && f >= -1 && f <= nx;
    double qR[7];
    if (has_nb) {
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double hi;
            recon_faces<LIM>(LIM == 2 ? sP[v][t - 2] : 0.0, sP[v][t - 1], q[v], sP[v][t + 1],
                             LIM == 2 ? sP[v][t + 2] : 0.0, qR[v], hi);
            sQ[v][t] = hi;
        }
    }
    __syncthreads();

    // Riemann problem on the lower face of cell f (faces 0 .. nx)
    const bool face = has_nb && t >= H && f >= 0;
    double F[7] = { 0, 0, 0, 0, 0, 0, 0 }, w = 0.5, uct[5];
    if (face) {
        Side L = { sQ[0][t - 1], sQ[1][t - 1], sQ[2][t - 1], sQ[3][t - 1], sQ[4][t - 1], sQ[5][t - 1], sQ[6][t - 1] };
        Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
        hlld_t<UCT>(L, R, bxf, g.gamma, g.igm1, F, w, uct);
        sP[0][t] = F[0]; sP[1][t] = F[1]; sP[2][t] = F[2]; sP[3][t] = F[3]; sP[4][t] = F[6];
        if (TWO_D) sP[5][t] = F[5];
    }
    __syncthreads();

    // cell f in [0, nx): flux difference with the right neighbour's face, CT data of the own face
    if (face && f < nx && t <= SX_NT - H - 1) {
        const double dtdx = P->dtdx[0];
        double r0 = fma(-dtdx, sP[0][t + 1] - F[0], rho);
        double r1 = fma(-dtdx, sP[1][t + 1] - F[1], mx);
        double r2 = fma(-dtdx, sP[2][t + 1] - F[2], my);
        double r3 = fma(-dtdx, sP[3][t + 1] - F[3], mz);
        double r4 = fma(-dtdx, sP[4][t + 1] - F[6], En);
        if (cb.Sn) {
            r0 = fma(cb.wn, o0, cb.ws * r0); r1 = fma(cb.wn, o1, cb.ws * r1); r2 = fma(cb.wn, o2, cb.ws * r2);
            r3 = fma(cb.wn, o3, cb.ws * r3); r4 = fma(cb.wn, o4, cb.ws * r4);
        }
        Sout[c] = r0; Sout[sa + c] = r1; Sout[2 * sa + c] = r2; Sout[3 * sa + c] = r3; Sout[4 * sa + c] = r4;
        if (TWO_D) {   // B_z has no faces in 2D: cell centred, flux updated
            double r7 = fma(-dtdx, sP[5][t + 1] - F[5], Bc[2]);
            Sout[7 * sa + c] = cb.Sn ? fma(cb.wn, o7, cb.ws * r7) : r7;
        }
        if (UCT) {
#pragma unroll
            for (int m = 0; m < 5; m++) uo.p[m][c] = uct[m];
            return;
        }
        // cell-centred EMF  E^c = -(v x B)
        const double e0 = q[3] * q[4] - q[2] * q[5], e1 = q[1] * q[5] - q[3] * Bc[0], e2 = q[2] * Bc[0] - q[1] * q[4];
        ct[(CT_FEM + 0) * sa + c] = F[4];
        ct[(CT_FEM + 1) * sa + c] = F[5];
        ct[(CT_W + 0) * sa + c] = w;
        ct[(CT_EC + 0) * sa + c] = e0;
        ct[(CT_EC + 1) * sa + c] = e1;
        ct[(CT_EC + 2) * sa + c] = e2;
        const int xdup = ct_xdup(f, nx);
        if (xdup) {
            const long long cd = c + xdup;
            ct[(CT_FEM + 0) * sa + cd] = F[4];
            ct[(CT_FEM + 1) * sa + cd] = F[5];
            ct[(CT_W + 0) * sa + cd] = w;
            ct[(CT_EC + 0) * sa + cd] = e0;
            ct[(CT_EC + 1) * sa + cd] = e1;
            ct[(CT_EC + 2) * sa + cd] = e2;
        }
    }
}

// ---------------------------------------------------------------- y / z sweep (a2-a5 fused), marching
// Thread = one column (fixed i and transverse index), marching along DIR over `seglen` cells.  It
// keeps the running q^L, the last two primitive states (as state + difference) and the previous
// flux in registers, so every cell is loaded and converted once and every flux is computed once per
// segment (+1 at the segment end).  The update is
//     Sout = base - scale * dt/dx_d * (F_d(+) - F_d(-)),  scale = 1 (Euler stage) or the combine weight ws,
// with base = Sout when the x+y sweep has already left its result there (update in place), or base = Sin
// when this sweep runs FIRST in a plain Euler stage and the x+y sweep then finishes the zone from Sout
// (the read-modify-write of S' moves from this HBM-bound kernel to the ALU-bound one).
// The operands of iteration s+1 travel global -> shared by 8-byte cp.async while interface s is
// being solved (two slots per thread, no block synchronisation: a thread only reads what it copied).

// cons -> rotated primitives of one cell (Eq. 7); B = cell-centred field
template <int DIR>
__device__ __forceinline__ void prim_rot(double rho, const double m[3], const double B[3], double En, double gamma,
                                         double q[7], bool &bad)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    double ir = rcp_fast(rho);
    // the velocities and the pressure are rounded products (__dmul_rn is never contracted into the
    // consumer's add): a zone's primitives are then the same bits wherever they are formed -- the first
    // cells of a march segment or the running loop -- and a run does not depend on how the marches are cut
    double v[3] = { __dmul_rn(m[0], ir), __dmul_rn(m[1], ir), __dmul_rn(m[2], ir) };
    double p = __dmul_rn(gamma - 1.0, fma(-0.5, fma(B[0], B[0], fma(B[1], B[1], B[2] * B[2])),
                                          fma(-0.5, fma(m[0], v[0], fma(m[1], v[1], m[2] * v[2])), En)));
    q[0] = rho; q[1] = v[DIR]; q[2] = v[T1]; q[3] = v[T2]; q[4] = B[T1]; q[5] = B[T2]; q[6] = p;
    bad = unphysical(rho) || unphysical(p);
}

template <int DIR, bool TWO_D>
__device__ __forceinline__ void load_rot(const Grid &g, const double *__restrict__ S, long long c, double q[7], bool &bad)
{
    const long long sa = g.sa;
    double m[3] = { S[sa + c], S[2 * sa + c], S[3 * sa + c] };
    double B[3];
    cell_b<TWO_D>(g, S + S_B * sa, c, B);
    prim_rot<DIR>(S[c], m, B, S[4 * sa + c], g.gamma, q, bad);
}

// 8-byte asynchronous global -> shared copy (LDGSTS)
__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int MARCH_NT = 128;
constexpr int MARCH_PF = 16;     // doubles per thread and iteration: U(s+1) 5, faces 5, U'(s-1) 6

// three blocks of 128 threads per SM: 168 registers per thread hold the running state without
// spilling (measured: 4 blocks at 128 registers spill ~40 values per interface and run 20% slower)
constexpr int MARCH_MINB = 3;
template <int DIR, int LIM, bool TWO_D, bool BOUND, bool UCT>
__global__ void __launch_bounds__(MARCH_NT, MARCH_MINB)
k_sweep_march(Grid g, const double *__restrict__ Sin, double *Sout, const double *base, double *__restrict__ ct,
              StepParams *P, double scale, int seglen, int tr0, BoundGrid bg, UctOut uo)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    constexpr bool BZ2D = TWO_D && DIR == 1;           // F_y[B_z] updates the cell-centred B_z in 2D
    __shared__ double pf[2][MARCH_PF][MARCH_NT];
    __shared__ double sbnd[BOUND ? 3 : 1][MARCH_NT];
    const int t = threadIdx.x;
    const int i = blockIdx.x * blockDim.x + t;
    if (i >= g.n[0]) return;
    // DIR = 1: grid.y = segment, grid.z = k;   DIR = 2: grid.y = j, grid.z = segment
    const int seg = DIR == 1 ? blockIdx.y : blockIdx.z;
    // transverse index; the y sweep of a 3D run also covers planes -1 and nz (tr0 = -1): the CT kernel
    // reads the y-face data one plane beyond the interior (no z wrap)
    const int tr = (DIR == 1 ? blockIdx.z : blockIdx.y) + tr0;
    const int s0 = seg * seglen;
    const int s1 = min(s0 + seglen, g.n[DIR]);
    // (the z sweep also leaves the CT data of the upper boundary face n: a periodic single domain gets
    // the same bits as on face 0; a z slab gets the face it shares with the slab above)
    const long long sa = g.sa, st = g.st[DIR];
    long long c = DIR == 1 ? g.at(i, s0, tr) : g.at(i, tr, s0);   // cell s0 of the segment
    const double gamma = g.gamma, igm1 = g.igm1;
    const double fac = scale * P->dtdx[DIR];
    const double *__restrict__ bn = Sin + (S_B + DIR) * sa;        // normal face field
    const double *__restrict__ b1 = Sin + (S_B + T1) * sa;         // transverse fields
    const double *__restrict__ b2 = Sin + (S_B + T2) * sa;
    const long long st1 = g.st[T1], st2 = g.st[T2];
    bool bad, anybad = false;
    SigmaBound sb;                                       // dt bound of the zones this thread finishes (last stage)
    if (BOUND) sb.init(&sbnd[0][t], MARCH_NT);

    // what iteration s consumes: U of cell s+1 and the faces around it, U' of cell s-1
    auto prefetch = [&](int slot, long long cs) {
        const long long cn = cs + st;                    // cell s+1
#pragma unroll
        for (int v = 0; v < 5; v++) cp_async8(&pf[slot][v][t], Sin + v * sa + cn);
        cp_async8(&pf[slot][5][t], bn + cn + st);        // upper normal face of cell s+1
        cp_async8(&pf[slot][6][t], b1 + cn);             // (2D: the cell-centred B_z itself)
        if (!(TWO_D && T1 == 2)) cp_async8(&pf[slot][7][t], b1 + cn + st1);
        cp_async8(&pf[slot][8][t], b2 + cn);
        if (!(TWO_D && T2 == 2)) cp_async8(&pf[slot][9][t], b2 + cn + st2);
        const long long cm = cs - st;
        cp_async8(&pf[slot][10][t], base + cm);
        cp_async8(&pf[slot][11][t], base + (1 + DIR) * sa + cm);
        cp_async8(&pf[slot][12][t], base + (1 + T1) * sa + cm);
        cp_async8(&pf[slot][13][t], base + (1 + T2) * sa + cm);
        cp_async8(&pf[slot][14][t], base + 4 * sa + cm);
        if (BZ2D) cp_async8(&pf[slot][15][t], base + 7 * sa + cm);
        cp_async_commit();
    };
    prefetch(0, c);

    // running state: q0 = primitives of cell s, d0 = q_s - q_{s-1}, qL = q^L of face s - 1/2,
    // Fp = flux through face s - 1/2 of the previous iteration, bface / bnext = b_n on faces s -+ 1/2
    double q0[7], d0[7], qL[7];
    {
        double qm[7];
        load_rot<DIR, TWO_D>(g, Sin, c - 2 * st, qm, bad);
        load_rot<DIR, TWO_D>(g, Sin, c - st, q0, bad);
#pragma unroll
        for (int v = 0; v < 7; v++) d0[v] = q0[v] - qm[v];
        load_rot<DIR, TWO_D>(g, Sin, c, qm, bad);           // qm now holds cell s0
        anybad |= bad;
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double d1 = qm[v] - q0[v], lo;
            plm_faces<LIM>(q0[v], d0[v], d1, lo, qL[v]);      // q^L of face s0 - 1/2
            q0[v] = qm[v];
            d0[v] = d1;
        }
    }
    double Fp[6] = { 0, 0, 0, 0, 0, 0 };                // previous face: rho, m_n, m_t1, m_t2, E, (B_z in 2D)
    double bface = bn[c];                               // normal field on face s - 1/2
    double bnext = bn[c + st];                          // ... on face s + 1/2

    // one interface; SLOT is the prefetch buffer holding the operands of this iteration
    auto iteration = [&](const int slot, const int s) {
        if (s < s1) { prefetch(slot ^ 1, c + st); cp_async_wait<1>(); }
        else        { cp_async_wait<0>(); }
        // cell s is in q0 (with d0 = q_s - q_{s-1}); cell s+1 arrives through shared memory
        double q1[7];
        const double bup = pf[slot][5][t];
        {
            double m[3], B[3];
            m[0] = pf[slot][1][t]; m[1] = pf[slot][2][t]; m[2] = pf[slot][3][t];
            B[DIR] = 0.5 * (bnext + bup);
            B[T1] = (TWO_D && T1 == 2) ? pf[slot][6][t] : 0.5 * (pf[slot][6][t] + pf[slot][7][t]);
            B[T2] = (TWO_D && T2 == 2) ? pf[slot][8][t] : 0.5 * (pf[slot][8][t] + pf[slot][9][t]);
            prim_rot<DIR>(pf[slot][0][t], m, B, pf[slot][4][t], gamma, q1, bad);
        }
        if (s + 1 < s1) anybad |= bad;
        Side L = { qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6] };
        double qR[7];
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double d1 = q1[v] - q0[v];
            plm_faces<LIM>(q0[v], d0[v], d1, qR[v], qL[v]);   // qL now carries the next q^L
            q0[v] = q1[v];
            d0[v] = d1;
        }
        Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
        double F[7], w, uct[5];
        hlld_t<UCT>(L, R, bface, gamma, igm1, F, w, uct);
        bface = bnext; bnext = bup;
        if (s > s0) {
            const long long cm = c - st;                  // cell s-1
            double m[3];
            const double r0 = fma(-fac, F[0] - Fp[0], pf[slot][10][t]);
            m[DIR] = fma(-fac, F[1] - Fp[1], pf[slot][11][t]);
            m[T1] = fma(-fac, F[2] - Fp[2], pf[slot][12][t]);
            m[T2] = fma(-fac, F[3] - Fp[3], pf[slot][13][t]);
            const double r4 = fma(-fac, F[6] - Fp[4], pf[slot][14][t]);
            Sout[cm] = r0;
            Sout[(1 + DIR) * sa + cm] = m[DIR];
            Sout[(1 + T1) * sa + cm] = m[T1];
            Sout[(1 + T2) * sa + cm] = m[T2];
            Sout[4 * sa + cm] = r4;
            if (BZ2D) Sout[7 * sa + cm] = fma(-fac, F[4] - Fp[5], pf[slot][15][t]);   // F_y[B_z]
            if (BOUND) sb.add(g, r0, m[0], m[1], m[2], r4);
        }
        if (UCT) {
            if (s < s1 || (DIR == 2 && s == g.n[2])) {
#pragma unroll
                for (int m = 0; m < 5; m++) uo.p[m][c] = uct[m];
            }
        } else if (s < s1 || (DIR == 2 && s == g.n[2])) {
            ct[(CT_FEM + 2 * DIR) * sa + c] = F[4];
            ct[(CT_FEM + 2 * DIR + 1) * sa + c] = F[5];
            ct[(CT_W + DIR) * sa + c] = w;
            const int xdup = ct_xdup(blockIdx.x * MARCH_NT + threadIdx.x, g.n[0]);
            if (xdup) {
                ct[(CT_FEM + 2 * DIR) * sa + c + xdup] = F[4];
                ct[(CT_FEM + 2 * DIR + 1) * sa + c + xdup] = F[5];
                ct[(CT_W + DIR) * sa + c + xdup] = w;
            }
        }
        Fp[0] = F[0]; Fp[1] = F[1]; Fp[2] = F[2]; Fp[3] = F[3]; Fp[4] = F[6]; Fp[5] = F[4];
        c += st;
    };
    // two interfaces per trip so that the running state needs no register rotation
    int s = s0;
    for (; s + 1 <= s1; s += 2) {
        iteration(0, s);
        iteration(1, s + 1);
    }
    if (s <= s1) iteration(0, s);
    if (anybad) P->err = 1;
    if (BOUND) bound_publish(bg, DIR == 1 ? s0 : tr, DIR == 1 ? tr : s0, sb.value(g, bg.cfac));
}

// ---------------------------------------------------------------- y / z sweep with the five-cell WENO-Z stencil
// Same marching scheme as k_sweep_march, for the reconstruction of [51] (reading R18):
// the primitives of cells s-2 .. s+2 live in a five-slot ring in shared memory (own column), iteration s
// reconstructs both faces of cell s, solves interface s - 1/2 with the q^L kept from cell s-1 and
// finishes cell s-1.  First version: operands are loaded directly (no prefetch ring).
constexpr int WZ_PF = 17;        // doubles per thread and iteration: U(s+3) 5, faces 6, U'(s) 6

template <int DIR, bool TWO_D, bool BOUND, bool UCT>
__global__ void __launch_bounds__(MARCH_NT, 3)
k_sweep_march_wz(Grid g, const double *__restrict__ Sin, double *Sout, double *__restrict__ ct, StepParams *P,
                 double scale, int seglen, int tr0, BoundGrid bg, UctOut uo)
{
    constexpr int T1 = (DIR + 1) % 3, T2 = (DIR + 2) % 3;
    constexpr bool BZ2D = TWO_D && DIR == 1;           // F_y[B_z] updates the cell-centred B_z in 2D
    extern __shared__ double wz_smem[];
    double (*ring)[7][MARCH_NT] = reinterpret_cast<double (*)[7][MARCH_NT]>(wz_smem);                    // [5]
    double (*pf)[WZ_PF][MARCH_NT] = reinterpret_cast<double (*)[WZ_PF][MARCH_NT]>(wz_smem + 5 * 7 * MARCH_NT);   // [2]
    __shared__ double sbnd[BOUND ? 3 : 1][MARCH_NT];
    const int t = threadIdx.x;
    const int i = blockIdx.x * blockDim.x + t;
    if (i >= g.n[0]) return;
    const int seg = DIR == 1 ? blockIdx.y : blockIdx.z;
    const int tr = (DIR == 1 ? blockIdx.z : blockIdx.y) + tr0;    // see k_sweep_march
    const int s0 = seg * seglen;
    const int s1 = min(s0 + seglen, g.n[DIR]);
    const long long sa = g.sa, st = g.st[DIR];
    long long c = DIR == 1 ? g.at(i, s0, tr) : g.at(i, tr, s0);   // cell s0 of the segment
    const double gamma = g.gamma, igm1 = g.igm1;
    const double fac = scale * P->dtdx[DIR];
    const double *__restrict__ bn = Sin + (S_B + DIR) * sa;        // normal face field
    const double *__restrict__ b1 = Sin + (S_B + T1) * sa;         // transverse fields
    const double *__restrict__ b2 = Sin + (S_B + T2) * sa;
    const long long st1 = g.st[T1], st2 = g.st[T2];
    const int xdup = ct_xdup(i, g.n[0]);
    bool bad, anybad = false;
    SigmaBound sb;
    if (BOUND) sb.init(&sbnd[0][t], MARCH_NT);
    auto slot = [](int m) { return ((m % 5) + 5) % 5; };

    // what iteration s consumes: U of cell s+2 and the faces around it, U' of cell s-1 (cs = cell s)
    auto prefetch = [&](int sl, long long cs) {
        const long long cn = cs + 2 * st;
#pragma unroll
        for (int v = 0; v < 5; v++) cp_async8(&pf[sl][v][t], Sin + v * sa + cn);
        cp_async8(&pf[sl][5][t], bn + cn);
        cp_async8(&pf[sl][6][t], bn + cn + st);
        cp_async8(&pf[sl][7][t], b1 + cn);               // (2D: the cell-centred B_z itself)
        if (!(TWO_D && T1 == 2)) cp_async8(&pf[sl][8][t], b1 + cn + st1);
        cp_async8(&pf[sl][9][t], b2 + cn);
        if (!(TWO_D && T2 == 2)) cp_async8(&pf[sl][10][t], b2 + cn + st2);
        const long long cm = cs - st;
        cp_async8(&pf[sl][11][t], Sout + cm);
        cp_async8(&pf[sl][12][t], Sout + (1 + DIR) * sa + cm);
        cp_async8(&pf[sl][13][t], Sout + (1 + T1) * sa + cm);
        cp_async8(&pf[sl][14][t], Sout + (1 + T2) * sa + cm);
        cp_async8(&pf[sl][15][t], Sout + 4 * sa + cm);
        if (BZ2D) cp_async8(&pf[sl][16][t], Sout + 7 * sa + cm);
        cp_async_commit();
    };
    prefetch(0, c);

    // prologue: cells s0-3 .. s0+1; q^L of face s0 - 1/2 comes from the stencil of cell s0-1
    double qL[7];
    {
        double w[5][7];
#pragma unroll
        for (int m = 0; m < 5; m++) {
            load_rot<DIR, TWO_D>(g, Sin, c + (m - 3) * st, w[m], bad);
            if (m >= 3 && s0 + m - 3 < s1) anybad |= bad;
        }
#pragma unroll
        for (int v = 0; v < 7; v++) {
            double lo;
            recon_faces<2>(w[0][v], w[1][v], w[2][v], w[3][v], w[4][v], lo, qL[v]);
        }
#pragma unroll
        for (int m = 1; m < 5; m++) {
            const int sl = slot(s0 + m - 3);
#pragma unroll
            for (int v = 0; v < 7; v++) ring[sl][v][t] = w[m][v];
        }
    }
    double Fp[6] = { 0, 0, 0, 0, 0, 0 };                // previous face: rho, m_n, m_t1, m_t2, E, (B_z in 2D)

    for (int s = s0; s <= s1; s++, c += st) {
        const int ps = (s - s0) & 1;
        if (s < s1) { prefetch(ps ^ 1, c + st); cp_async_wait<1>(); }
        else        { cp_async_wait<0>(); }
        {   // cell s+2 replaces cell s-3 in the ring
            double qa[7], m[3], B[3];
            m[0] = pf[ps][1][t]; m[1] = pf[ps][2][t]; m[2] = pf[ps][3][t];
            B[DIR] = 0.5 * (pf[ps][5][t] + pf[ps][6][t]);
            B[T1] = (TWO_D && T1 == 2) ? pf[ps][7][t] : 0.5 * (pf[ps][7][t] + pf[ps][8][t]);
            B[T2] = (TWO_D && T2 == 2) ? pf[ps][9][t] : 0.5 * (pf[ps][9][t] + pf[ps][10][t]);
            prim_rot<DIR>(pf[ps][0][t], m, B, pf[ps][4][t], gamma, qa, bad);
            if (s + 2 < s1) anybad |= bad;
            const int sl = slot(s + 2);
#pragma unroll
            for (int v = 0; v < 7; v++) ring[sl][v][t] = qa[v];
        }
        const int m2 = slot(s - 2), m1 = slot(s - 1), c0 = slot(s), p1 = slot(s + 1), p2 = slot(s + 2);
        double qR[7], qLn[7];
#pragma unroll
        for (int v = 0; v < 7; v++)
            recon_faces<2>(ring[m2][v][t], ring[m1][v][t], ring[c0][v][t], ring[p1][v][t], ring[p2][v][t], qR[v], qLn[v]);
        Side L = { qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6] };
        Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
        double F[7], w, uct[5];
        hlld_t<UCT>(L, R, bn[c], gamma, igm1, F, w, uct);
#pragma unroll
        for (int v = 0; v < 7; v++) qL[v] = qLn[v];
        if (s > s0) {
            const long long cm = c - st;                  // cell s-1
            double m[3];
            const double r0 = fma(-fac, F[0] - Fp[0], pf[ps][11][t]);
            m[DIR] = fma(-fac, F[1] - Fp[1], pf[ps][12][t]);
            m[T1] = fma(-fac, F[2] - Fp[2], pf[ps][13][t]);
            m[T2] = fma(-fac, F[3] - Fp[3], pf[ps][14][t]);
            const double r4 = fma(-fac, F[6] - Fp[4], pf[ps][15][t]);
            Sout[cm] = r0;
            Sout[(1 + DIR) * sa + cm] = m[DIR];
            Sout[(1 + T1) * sa + cm] = m[T1];
            Sout[(1 + T2) * sa + cm] = m[T2];
            Sout[4 * sa + cm] = r4;
            if (BZ2D) Sout[7 * sa + cm] = fma(-fac, F[4] - Fp[5], pf[ps][16][t]);   // F_y[B_z]
            if (BOUND) sb.add(g, r0, m[0], m[1], m[2], r4);
        }
        if (UCT) {
            if (s < s1 || (DIR == 2 && s == g.n[2])) {
#pragma unroll
                for (int m = 0; m < 5; m++) uo.p[m][c] = uct[m];
            }
        } else if (s < s1 || (DIR == 2 && s == g.n[2])) {
            ct[(CT_FEM + 2 * DIR) * sa + c] = F[4];
            ct[(CT_FEM + 2 * DIR + 1) * sa + c] = F[5];
            ct[(CT_W + DIR) * sa + c] = w;
            if (xdup) {
                ct[(CT_FEM + 2 * DIR) * sa + c + xdup] = F[4];
                ct[(CT_FEM + 2 * DIR + 1) * sa + c + xdup] = F[5];
                ct[(CT_W + DIR) * sa + c + xdup] = w;
            }
        }
        Fp[0] = F[0]; Fp[1] = F[1]; Fp[2] = F[2]; Fp[3] = F[3]; Fp[4] = F[6]; Fp[5] = F[4];
    }
    if (anybad) P->err = 1;
    if (BOUND) bound_publish(bg, DIR == 1 ? s0 : tr, DIR == 1 ? tr : s0, sb.value(g, bg.cfac));
}
constexpr int WZ_SMEM_BYTES = (5 * 7 + 2 * WZ_PF) * MARCH_NT * 8;

// ---------------------------------------------------------------- fused x + y sweep (a2-a5)
// Block = NT consecutive cells of one x-row, marching along y over `seglen` rows.  Each arriving row
// is converted to primitives once and kept in a three-row ring in shared memory.  The x interfaces of
// a row are solved across the block (q^L and the fluxes are exchanged through shared memory, as in
// k_sweep_x); the y interfaces are solved down each thread's own column from the ring (as in
// k_sweep_march).  A cell is therefore read once and written once for both directions:
//     S' = (S - dt/dx (Fx(+) - Fx(-))) - dt/dy (Fy(+) - Fy(-))      [combine: wn S^n + ws S']
// WRAP: the block spans the whole periodic row (NT = nx), neighbours wrap inside shared memory and
// no lane is idle.  Otherwise blocks overlap by four cells like k_sweep_x.
// Operands travel global -> shared as whole row segments by TMA bulk copies (cp.async.bulk + mbarrier)
// issued by one thread: group A, the row that arrives next, one iteration ahead; group F, S and S^n of
// the row that is finished in this iteration.  They bypass L1 and cost the other threads no instruction.
// fin: the state the finished row starts from -- Sin, or Sout when the z sweep has already run in this
// stage and left S - dt/dz (Fz(+) - Fz(-)) there (see k_sweep_march).
constexpr int XY_RING = 9;       // rho, vx, vy, vz, Bx, By, Bz, p (cell centred), b_x on the lower x-face
constexpr int XY_PFA = 10;       // arriving row: U 5, (rows 5, 6: carried y flux, see fpy), by upper 7, bz 8, bz upper 9
constexpr int XY_PFF = 11;       // finishing row: U 5, S^n 6
constexpr int XY_DOUBLES_PER_THREAD = 3 * XY_RING + XY_PFA + XY_PFF + 7;
constexpr int XY_BXROW_PAD = 2;     // the b_x row of the arriving row holds NT + 2 faces (thread t reads faces t, t + 1)
constexpr int XY_SMEM_EXTRA(int nt) { return (nt + XY_BXROW_PAD) * 8 + 32; }   // b_x row + three mbarriers behind the arrays

// 128-thread blocks run three per SM at 168 registers (measured 17% faster than four at 128)
constexpr int XY128_MINB = 3;
// UCT: UCT-HLLD mode (R19): the five face numbers of hlld_t<true> go to ux / uy instead of the CT arrays.
template <int LIM, bool TWO_D, bool WRAP, int NT, bool UCT>
__global__ void __launch_bounds__(NT, NT == 128 ? XY128_MINB : 512 / NT)
k_sweep_xy(Grid g, const double *__restrict__ Sin, double *Sout, const double *fin, double *__restrict__ ct,
           StepParams *P, Combine cb, int seglen, int kz0, UctOut ux, UctOut uy)
{
    extern __shared__ __align__(128) double xy_smem[];
    const int t = threadIdx.x;
    double *ring = xy_smem;                       // [3][XY_RING][NT]
    double *pfa = ring + 3 * XY_RING * NT;        // [XY_PFA][NT]
    double *pff = pfa + XY_PFA * NT;              // [XY_PFF][NT]
    double *sQ = pff + XY_PFF * NT;               // [7][NT]: q^L along x, then the x fluxes
    double *bxrow = sQ + 7 * NT;                  // [NT + 2]: b_x faces of the arriving row
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(bxrow + NT + XY_BXROW_PAD);   // [3]: group A, group F, x fluxes
    // The previous y flux is needed again only when its row is finished, a whole iteration later: its
    // first components wait in otherwise unused shared-memory rows instead of registers (which would
    // be spilled to local memory): pfa rows 5 and 6, and in 3D the sQ rows 5 and 6 that only 2D uses.
    constexpr int NFPS = TWO_D ? 2 : 4;
    double *const fpy[4] = { pfa + 5 * NT + t, pfa + 6 * NT + t, sQ + 5 * NT + t, sQ + 6 * NT + t };
    const int nx = g.n[0];
    const int i = WRAP ? t : (int)blockIdx.x * (NT - 4) - 2 + t;
    const bool valid = WRAP || i < nx + 2;
    const int tl = WRAP ? (t == 0 ? NT - 1 : t - 1) : max(t - 1, 0);
    const int tr = WRAP ? (t == NT - 1 ? 0 : t + 1) : min(t + 1, NT - 1);
    const bool has_slope = WRAP || (valid && t >= 1 && t <= NT - 2 && i + 1 < nx + 2);
    const bool xface = WRAP || (has_slope && t >= 2 && i <= nx);
    const bool cell = WRAP || (xface && t <= NT - 3 && i < nx);     // this thread owns an interior cell
    const int xdup = cell ? ct_xdup(i, nx) : 0;
    // only the warps holding the first / last cell of the row write periodic copies: a warp-uniform branch
    // spares the other warps the predicated stores
    const bool wdup = __any_sync(0xffffffffu, xdup != 0);
    // 3D: kz0 = -1 and the grid covers planes -1 .. nz: the CT kernel reads the x- and y-face data one plane
    // beyond the interior (no z wrap: a z slab's neighbour planes are not its own).  Only the CT data of
    // those two planes is used; their hydro update lands in ghost planes of Sout, which nothing reads
    // before the next ghost fill overwrites them.
    const int k = (int)blockIdx.z + kz0;
    const int s0 = blockIdx.y * seglen, s1 = min(s0 + seglen, g.n[1]);
    const long long sa = g.sa, st = g.st[1], stz = g.st[2];
    const double gamma = g.gamma;
    const double dtdx = P->dtdx[0];
    const bool combine = cb.Sn != nullptr;
    const double facy = (combine ? cb.ws : 1.0) * P->dtdx[1];
    const double *__restrict__ bx = Sin + S_B * sa;
    const double *__restrict__ by = Sin + (S_B + 1) * sa;
    const double *__restrict__ bz = Sin + (S_B + 2) * sa;
    long long c = g.at(valid ? i : 0, s0, k);                       // cell (i, s0, k)
    bool anybad = false;

    // TMA row copies, issued by thread 0: the block's x range [i0, i0 + NT) of one row of each array
    const long long row0 = g.at(WRAP ? 0 : (int)blockIdx.x * (NT - 4) - 2, s0, k);    // first cell of row s0
    constexpr unsigned ROWB = NT * 8;
    auto issue_arrive = [&](long long cr) {                         // cr = first cell of the arriving row
        mbar_expect_tx(bars, (TWO_D ? 8 : 9) * ROWB + 16);
#pragma unroll
        for (int v = 0; v < 5; v++) tma_bulk_g2s(pfa + v * NT, Sin + v * sa + cr, ROWB, bars);
        tma_bulk_g2s(bxrow, bx + cr, ROWB + 16, bars);                // NT + 2 faces: thread t also reads face t + 1
        tma_bulk_g2s(pfa + 7 * NT, by + cr + st, ROWB, bars);
        tma_bulk_g2s(pfa + 8 * NT, bz + cr, ROWB, bars);
        if (!TWO_D) tma_bulk_g2s(pfa + 9 * NT, bz + cr + stz, ROWB, bars);
    };
    auto issue_finish = [&](long long cf) {                         // cf = first cell of the row finished next
        mbar_expect_tx(bars + 1, (5 + (combine ? (TWO_D ? 6 : 5) : 0)) * ROWB);
#pragma unroll
        for (int v = 0; v < 5; v++) tma_bulk_g2s(pff + v * NT, fin + v * sa + cf, ROWB, bars + 1);
        if (combine) {
#pragma unroll
            for (int v = 0; v < 5; v++) tma_bulk_g2s(pff + (5 + v) * NT, cb.Sn + v * sa + cf, ROWB, bars + 1);
            if (TWO_D) tma_bulk_g2s(pff + 10 * NT, cb.Sn + 7 * sa + cf, ROWB, bars + 1);
        }
    };
    if (t == 0) {
        mbar_init(bars, 1);
        mbar_init(bars + 1, 1);
        mbar_init(bars + 2, NT / 32);                               // one arrival per warp
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (t == 0) issue_arrive(row0 + st);                            // group A(s0): row s0 + 1
    // primitives of one cell from its conserved variables and the faces around it
    auto to_prim = [&](double rho, double mx, double my, double mz, double En, double B0, double B1, double B2,
                       double q[8], bool &bad) {
        double ir = rcp_fast(rho);
        q[0] = rho; q[1] = __dmul_rn(mx, ir); q[2] = __dmul_rn(my, ir); q[3] = __dmul_rn(mz, ir);      // see prim_rot
        q[4] = B0; q[5] = B1; q[6] = B2;
        q[7] = __dmul_rn(gamma - 1.0, fma(-0.5, fma(B0, B0, fma(B1, B1, B2 * B2)),
                                          fma(-0.5, fma(mx, q[1], fma(my, q[2], mz * q[3])), En)));
        bad = unphysical(rho) || unphysical(q[7]);
    };
    auto load_prim = [&](long long cc, double q[8], double &bxf, bool &bad) {
        double B[3];
        cell_b<TWO_D>(g, bx, cc, B);
        bxf = bx[cc];
        to_prim(Sin[cc], Sin[sa + cc], Sin[2 * sa + cc], Sin[3 * sa + cc], Sin[4 * sa + cc], B[0], B[1], B[2], q, bad);
    };

    // ---- prologue: rows s0-2, s0-1, s0 straight from global; s0-1 and s0 enter the ring
    double qLy[7];                                   // y-rotated q^L of face s - 1/2: rho, vy, vz, vx, Bz, Bx, p
    double bface, bnext;                             // b_y on faces s - 1/2 and s + 1/2
    {
        double qa[8], qb[8], qc[8], f0, f1, f2;
        bool bad;
        if (valid) {
            load_prim(c - 2 * st, qa, f0, bad);
            load_prim(c - st, qb, f1, bad);
            load_prim(c, qc, f2, bad);
            if (cell) anybad |= bad;
            bface = by[c]; bnext = by[c + st];
        } else {
#pragma unroll
            for (int v = 0; v < 8; v++) { qa[v] = qb[v] = qc[v] = (v == 0 || v == 7) ? 1.0 : 0.0; }
            f1 = f2 = 0.0; bface = bnext = 0.0;
        }
        const int rot[7] = { 0, 2, 3, 1, 6, 4, 7 };
#pragma unroll
        for (int v = 0; v < 7; v++) {
            const int r = rot[v];
            qLy[v] = qb[r] + 0.5 * plm_slope<LIM>(qb[r] - qa[r], qc[r] - qb[r]);
        }
        double *rb = ring + t, *rc = ring + XY_RING * NT + t;
#pragma unroll
        for (int v = 0; v < 8; v++) { rb[v * NT] = qb[v]; rc[v * NT] = qc[v]; }
        rb[8 * NT] = f1; rc[8 * NT] = f2;
    }
    double Fpy[6] = { 0, 0, 0, 0, 0, 0 };            // previous y-face: rho, m_y, m_z, m_x, E, (B_z in 2D);
                                                     // components < NFPS live in shared memory (fpy)
    // ring rows s-1, s, s+1 (own column; neighbours at +-1): the three slots rotate every iteration
    double *rm = ring + t, *r0 = ring + XY_RING * NT + t, *rn = ring + 2 * XY_RING * NT + t;
    const int dl = tl - t, dr = tr - t;
    const int dll = (WRAP ? (t >= 2 ? t - 2 : t - 2 + NT) : max(t - 2, 0)) - t;

    for (int s = s0; s <= s1; s++, c += st) {
        // ---- (1) the arriving row s+1: convert, ring
        mbar_wait(bars, (s - s0) & 1);               // group A(s) has landed
        double q1[8], byu = 0.0;
        {
            bool bad = false;
            double bxf = 0.0;
            if (valid) {
                double B0 = 0.5 * (bxrow[t] + bxrow[t + 1]);
                byu = pfa[7 * NT + t];
                double B1 = 0.5 * (bnext + byu);
                double B2 = TWO_D ? pfa[8 * NT + t] : 0.5 * (pfa[8 * NT + t] + pfa[9 * NT + t]);
                bxf = bxrow[t];
                to_prim(pfa[t], pfa[NT + t], pfa[2 * NT + t], pfa[3 * NT + t], pfa[4 * NT + t], B0, B1, B2, q1, bad);
                if (cell && s + 1 < s1) anybad |= bad;
            } else {
#pragma unroll
                for (int v = 0; v < 8; v++) q1[v] = (v == 0 || v == 7) ? 1.0 : 0.0;
            }
#pragma unroll
            for (int v = 0; v < 8; v++) rn[v * NT] = q1[v];
            rn[8 * NT] = bxf;
        }
        __syncthreads();                             // B1: sQ free; everybody has read group A(s) and finished row s-2;
                                                     //     ring row s-1 and its neighbours are visible
        if (t == 0) {
            fence_proxy_async();
            const long long cr = row0 + (long long)(s - s0) * st;              // first cell of row s
            if (s < s1) issue_arrive(cr + 2 * st);                              // group A(s+1): row s + 2
            if (s > s0) issue_finish(cr - st);                                  // group F(s): row s - 1
        }

        // ---- (2) x interfaces of row s-1; their flux difference goes straight into the prefetched S of
        //      that row (group F(s), in shared memory), so nothing of it stays live across the y solve
        if (s > s0) {
            // Each thread limits the slopes of its own cell and of its left neighbour (whose q^L it
            // needs): 7 more slope evaluations than an exchange of q^L through shared memory, but two
            // block barriers and 14 shared-memory accesses fewer.
            const int xv[7] = { 0, 1, 2, 3, 5, 6, 7 };              // rho, vx, vy, vz, By, Bz, p
            double qR[7], qL[7], qo[8];
#pragma unroll
            for (int v = 0; v < 8; v++) qo[v] = rm[v * NT];
            if (xface) {
#pragma unroll
                for (int v = 0; v < 7; v++) {
                    const int r = xv[v];
                    const double q1m = rm[r * NT + dl], q2m = rm[r * NT + dll], q1p = rm[r * NT + dr];
                    double lo, hi;
                    plm_faces<LIM>(qo[r], qo[r] - q1m, q1p - qo[r], qR[v], hi);
                    plm_faces<LIM>(q1m, q1m - q2m, qo[r] - q1m, lo, qL[v]);
                }
            }
            Side L = { qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6] };
            double F[7] = { 0, 0, 0, 0, 0, 0, 0 }, w = 0.5, uctx[5] = { 0.5, 0, 0, 0, 0 };
            if (xface) {
                Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
                hlld_t<UCT>(L, R, rm[8 * NT], gamma, g.igm1, F, w, uctx);
                sQ[t] = F[0]; sQ[NT + t] = F[1]; sQ[2 * NT + t] = F[2]; sQ[3 * NT + t] = F[3]; sQ[4 * NT + t] = F[6];
                if (TWO_D) sQ[5 * NT + t] = F[5];
            }
            if (UCT) {
                if (cell) {
                    const long long cm = c - st;
#pragma unroll
                    for (int m = 0; m < 5; m++) ux.p[m][cm] = uctx[m];
                }
            } else if (cell) {
                const long long cm = c - st;
                // cell-centred EMF  E^c = -(v x B)
                const double e0 = qo[3] * qo[5] - qo[2] * qo[6], e1 = qo[1] * qo[6] - qo[3] * qo[4],
                             e2 = qo[2] * qo[4] - qo[1] * qo[5];
                ct[(CT_FEM + 0) * sa + cm] = F[4];
                ct[(CT_FEM + 1) * sa + cm] = F[5];
                ct[(CT_W + 0) * sa + cm] = w;
                ct[(CT_EC + 0) * sa + cm] = e0;
                ct[(CT_EC + 1) * sa + cm] = e1;
                ct[(CT_EC + 2) * sa + cm] = e2;
                if (wdup && xdup) {
                    const long long cd = cm + xdup;
                    ct[(CT_FEM + 0) * sa + cd] = F[4];
                    ct[(CT_FEM + 1) * sa + cd] = F[5];
                    ct[(CT_W + 0) * sa + cd] = w;
                    ct[(CT_EC + 0) * sa + cd] = e0;
                    ct[(CT_EC + 1) * sa + cd] = e1;
                    ct[(CT_EC + 2) * sa + cd] = e2;
                }
            }
            // split-phase barrier instead of a __syncthreads: every warp signals that its fluxes are in
            // shared memory and goes on to the y solve; the neighbour's flux is read only when the row is
            // finished, by which time every warp has long arrived (no waiting for the slowest x solve)
            __syncwarp();
            if ((t & 31) == 0) mbar_arrive(bars + 2);
        }

        // ---- (3) y interface s - 1/2 down the own column
        double Fy[7] = { 0, 0, 0, 0, 0, 0, 0 }, wy = 0.5;
        {
            const int rot[7] = { 0, 2, 3, 1, 6, 4, 7 };              // rho, vy, vz, vx, Bz, Bx, p
            double qR[7], nl[7];
#pragma unroll
            for (int v = 0; v < 7; v++) {
                const int r = rot[v];
                double qs = r0[r * NT];
                plm_faces<LIM>(qs, qs - rm[r * NT], rn[r * NT] - qs, qR[v], nl[v]);
            }
            if (cell) {
                Side L = { qLy[0], qLy[1], qLy[2], qLy[3], qLy[4], qLy[5], qLy[6] };
                Side R = { qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6] };
                double ucty[5];
                hlld_t<UCT>(L, R, bface, gamma, g.igm1, Fy, wy, ucty);
                if (UCT && s < s1) {
#pragma unroll
                    for (int m = 0; m < 5; m++) uy.p[m][c] = ucty[m];
                }
            }
#pragma unroll
            for (int v = 0; v < 7; v++) qLy[v] = nl[v];
        }

        // ---- (4) finish row s-1; CT data of the y face
        if (s > s0) {
            mbar_wait(bars + 2, (s - s0 - 1) & 1);   // all x fluxes of row s-1 are in shared memory
            mbar_wait(bars + 1, (s - s0 - 1) & 1);   // group F(s) has landed
        }
        if (s > s0 && cell) {
            const long long cm = c - st;
            // S of row s-1 minus the x flux difference (own lower face, right neighbour's lower face)
            double r0v = fma(-dtdx, sQ[tr] - sQ[t], pff[t]);
            double r1v = fma(-dtdx, sQ[NT + tr] - sQ[NT + t], pff[NT + t]);
            double r2v = fma(-dtdx, sQ[2 * NT + tr] - sQ[2 * NT + t], pff[2 * NT + t]);
            double r3v = fma(-dtdx, sQ[3 * NT + tr] - sQ[3 * NT + t], pff[3 * NT + t]);
            double r4v = fma(-dtdx, sQ[4 * NT + tr] - sQ[4 * NT + t], pff[4 * NT + t]);
            if (combine) {
                r0v = fma(cb.wn, pff[5 * NT + t], cb.ws * r0v); r1v = fma(cb.wn, pff[6 * NT + t], cb.ws * r1v);
                r2v = fma(cb.wn, pff[7 * NT + t], cb.ws * r2v); r3v = fma(cb.wn, pff[8 * NT + t], cb.ws * r3v);
                r4v = fma(cb.wn, pff[9 * NT + t], cb.ws * r4v);
            }
            // y-rotated flux: (rho, m_y, m_z, m_x, B_z, B_x, E)
#pragma unroll
            for (int n = 0; n < NFPS; n++) Fpy[n] = *fpy[n];
            r0v = fma(-facy, Fy[0] - Fpy[0], r0v);
            r2v = fma(-facy, Fy[1] - Fpy[1], r2v);
            r3v = fma(-facy, Fy[2] - Fpy[2], r3v);
            r1v = fma(-facy, Fy[3] - Fpy[3], r1v);
            r4v = fma(-facy, Fy[6] - Fpy[4], r4v);
            Sout[cm] = r0v;
            Sout[2 * sa + cm] = r2v;
            Sout[3 * sa + cm] = r3v;
            Sout[sa + cm] = r1v;
            Sout[4 * sa + cm] = r4v;
            if (TWO_D) {
                double r7v = fma(-dtdx, sQ[5 * NT + tr] - sQ[5 * NT + t], rm[6 * NT]);
                if (combine) r7v = fma(cb.wn, pff[10 * NT + t], cb.ws * r7v);
                Sout[7 * sa + cm] = fma(-facy, Fy[4] - Fpy[5], r7v);
            }
        }
        if (!UCT && cell && s < s1) {
            ct[(CT_FEM + 2) * sa + c] = Fy[4];
            ct[(CT_FEM + 3) * sa + c] = Fy[5];
            ct[(CT_W + 1) * sa + c] = wy;
            if (wdup && xdup) {
                ct[(CT_FEM + 2) * sa + c + xdup] = Fy[4];
                ct[(CT_FEM + 3) * sa + c + xdup] = Fy[5];
                ct[(CT_W + 1) * sa + c + xdup] = wy;
            }
        }
        {
            const double nf[6] = { Fy[0], Fy[1], Fy[2], Fy[3], Fy[6], Fy[4] };
#pragma unroll
            for (int n = 0; n < 6; n++) { if (n < NFPS) *fpy[n] = nf[n]; else Fpy[n] = nf[n]; }
        }
        bface = bnext; bnext = byu;
        double *rt = rm; rm = r0; r0 = rn; rn = rt;
    }
    if (anybad) P->err = 1;
}

// ---------------------------------------------------------------- CT (a6, R6) [+ RK2 combine of the faces (a7)]
// Edge EMF at the lower (A,B) edge of a cell (component EC, A = EC+1, B = EC+2 cyclic): arithmetic
// mean of the four face EMFs plus the upwinded half-cell differences to the cell-centred EMFs.
//   Ea_lo, Ea_hi : EMF on the two A-faces meeting at the edge (cells at B-1 and B)
//   Eb_lo, Eb_hi : EMF on the two B-faces (cells at A-1 and A)
//   wa_*, wb_*   : upwind weights on those faces
//   e00, e10, e01, e11 : cell EMFs of (A-1,B-1), (A,B-1), (A-1,B), (A,B)
__device__ __forceinline__ double edge_emf(double Ea_lo, double Ea_hi, double Eb_lo, double Eb_hi,
                                           double wa_lo, double wa_hi, double wb_lo, double wb_hi,
                                           double e00, double e10, double e01, double e11)
{
    // up(w; a, b) = w a + (1 - w) b = b + w (a - b)
    const double a1 = Eb_lo - e00, b1 = Eb_hi - e10, a2 = e01 - Eb_lo, b2 = e11 - Eb_hi;
    const double a3 = Ea_lo - e00, b3 = Ea_hi - e01, a4 = e10 - Ea_lo, b4 = e11 - Ea_hi;
    const double t1 = fma(wa_lo, a1 - b1, b1), t2 = fma(wa_hi, a2 - b2, b2);
    const double t3 = fma(wb_lo, a3 - b3, b3), t4 = fma(wb_hi, a4 - b4, b4);
    return 0.25 * (((Ea_lo + Ea_hi) + (Eb_lo + Eb_hi)) + ((t1 - t2) + (t3 - t4)));
}

// Block = CT_TX x CT_TY columns marching along z over `seglen` planes (k = k0 .. k1; the CT data of
// planes k0 - 1 and k1 is read too: -1 and nz lie in the ghost planes, written by the sweeps).  Iteration k forms
// E_z(i-1/2, j-1/2, k) and, from plane k and the plane k-1 values kept in registers, E_x(i, j-1/2, k-1/2)
// and E_y(i-1/2, j, k-1/2): 12 loads of the thread's own cell (HBM; prefetched into L2 one plane
// ahead) and 13 of its x-1 / y-1 neighbours (L1 hits: the neighbour thread loads the same words).
// The three EMFs are exchanged through shared memory (one barrier, double buffered) and the faces
// b_z(k), b_x(k-1), b_y(k-1) are updated with  db/dt = -curl E  (COMBINE: bout <- (bout + that)/2
// in place, bout holding the faces of S^n).  No edge EMF is ever stored in HBM.  Tiles overlap by
// one column and one row: the threads of the last column / row only supply the edges just outside
// the tile, so all threads run the same code and each face is written exactly once.
constexpr int CT_TX = 32, CT_TY = 8;

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <bool COMBINE, bool TWO_D>
__global__ void __launch_bounds__(CT_TX * CT_TY, 3)
k_ct(Grid g, const double *__restrict__ ct, const double *__restrict__ bin, double *bout,
     const StepParams *__restrict__ P, int seglen, double *__restrict__ dbg, Combine cb)
{
    __shared__ double sE[2][3][CT_TY][CT_TX];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int i = blockIdx.x * (CT_TX - 1) + tx, j = blockIdx.y * (CT_TY - 1) + ty;
    // cells i <= n0, j <= n1 supply edges (index n wraps to 0); faces are updated by the inner threads
    const bool edge = i <= g.n[0] && j <= g.n[1];
    const bool upd = tx < CT_TX - 1 && ty < CT_TY - 1 && i < g.n[0] && j < g.n[1];
    const int k0 = blockIdx.z * seglen, k1 = min(k0 + seglen, g.n[2]);
    const long long sa = g.sa, st2 = g.st[2];
    const double dtdx = P->dtdx[0], dtdy = P->dtdx[1], dtdz = P->dtdx[2];

    // clamp the indices of idle threads so that every address below is legal
    const int ii = edge ? (i == g.n[0] ? 0 : i) : 0, jj = edge ? (j == g.n[1] ? 0 : j) : 0;
    const int im = wrap_m1(ii, g.n[0]), jm = wrap_m1(jj, g.n[1]);
    const long long r0 = (long long)(jj + g.off[1]) * g.st[1] + g.off[0];
    const long long rm = (long long)(jm + g.off[1]) * g.st[1] + g.off[0];
    const long long oc = r0 + ii;                                      // own cell, in-plane offset
    const int XM = (int)(r0 + im - oc), YM = (int)(rm + ii - oc), XYM = (int)(rm + im - oc);   // neighbours
    // no z wrap: the sweeps leave the CT data of planes -1 and nz (and of the z face nz) as well
    auto plane = [&](int k) { return (long long)(k + g.off[2]) * st2; };
    // the CT arrays: F_x[By] 0, F_x[Bz] 1, F_y[Bz] 2, F_y[Bx] 3, F_z[Bx] 4, F_z[By] 5, w_x 6, w_y 7, w_z 8, E^c 9-11
    const double *__restrict__ A0 = ct + oc;

    // plane k-1 values that enter E_x, E_y at k - 1/2
    double fyz = 0, wyP = 0, excP = 0, excPm = 0, fxz = 0, wxP = 0, eycP = 0, eycPm = 0;
    if (!TWO_D) {
        const double *q = A0 + plane(k0 - 1);
        fyz = q[2 * sa];  wyP = q[7 * sa];
        excP = q[9 * sa]; excPm = q[9 * sa + YM];
        fxz = q[1 * sa];  wxP = q[6 * sa];
        eycP = q[10 * sa]; eycPm = q[10 * sa + XM];
    }
    double exP = 0.0, eyP = 0.0, dEzx = 0.0, dEzy = 0.0;
    // faces to update next: b_z(k), b_x(k-1), b_y(k-1) (+ the S^n faces in the combine stage)
    double pbx = 0, pby = 0, pbz = 0, qbx = 0, qby = 0, qbz = 0;
    if (upd) {
        const long long c = plane(k0) + oc;
        if (TWO_D) {
            pbx = bin[c]; pby = bin[sa + c];
            if (COMBINE) { qbx = cb.Sn[c]; qby = cb.Sn[sa + c]; }
        } else {
            pbz = bin[2 * sa + c];
            if (COMBINE) qbz = cb.Sn[2 * sa + c];
        }
    }
    for (int k = k0; k <= (TWO_D ? k0 : k1); k++) {
        const int buf = k & 1;
        const double *__restrict__ v = A0 + plane(k);
        if (!TWO_D && k + 1 <= k1) {                                   // own words of the next plane -> L2
            const double *q = A0 + plane(k + 1);
#pragma unroll
            for (int a = 0; a < CT_COUNT; a++) prefetch_l2(q + a * sa);
        }
        auto S = [&](int a, int off) { return v[a * sa + off]; };
        const double wx = S(6, 0), wy = S(7, 0);
        // E_z(i-1/2, j-1/2, k): A = x, B = y
        const double ez = edge_emf(-S(0, YM), -S(0, 0), S(3, XM), S(3, 0), S(6, YM), wx, S(7, XM), wy,
                                   S(11, XYM), S(11, YM), S(11, XM), S(11, 0));
        double exN = 0.0, eyN = 0.0;
        sE[buf][0][ty][tx] = ez;
        if (!TWO_D) {
            const double wz = S(8, 0);
            // E_x(i, j-1/2, k-1/2): A = y, B = z
            const double fyzN = S(2, 0), excN = S(9, 0), excNm = S(9, YM);
            exN = edge_emf(-fyz, -fyzN, S(5, YM), S(5, 0), wyP, wy, S(8, YM), wz, excPm, excP, excNm, excN);
            // E_y(i-1/2, j, k-1/2): A = z, B = x
            const double fxzN = S(1, 0), eycN = S(10, 0), eycNm = S(10, XM);
            eyN = edge_emf(-S(4, XM), -S(4, 0), fxz, fxzN, S(8, XM), wz, wxP, wx, eycPm, eycNm, eycP, eycN);
            sE[buf][1][ty][tx] = exN; sE[buf][2][ty][tx] = eyN;
            fyz = fyzN; wyP = wy; excP = excN; excPm = excNm;
            fxz = fxzN; wxP = wx; eycP = eycN; eycPm = eycNm;
        }
        __syncthreads();                                      // edge EMFs of this iteration are visible
        if (upd) {
            const double ezx = sE[buf][0][ty][tx + 1], ezy = sE[buf][0][ty + 1][tx];
            const long long c = plane(k) + oc;
            if (TWO_D) {
                const double bxn = fma(-dtdy, ezy - ez, pbx);
                const double byn = fma(dtdx, ezx - ez, pby);
                const double bxo = COMBINE ? fma(cb.wn, qbx, cb.ws * bxn) : bxn;
                bout[c] = bxo;
                if (i == 0) bout[c + g.n[0]] = bxo;       // periodic copy: x-face n0 is face 0
                bout[sa + c] = COMBINE ? fma(cb.wn, qby, cb.ws * byn) : byn;
                if (dbg) { dbg[c] = 0.0; dbg[sa + c] = 0.0; dbg[2 * sa + c] = ez; }
            } else {
                if (k > k0) {                                 // b_x, b_y of plane k-1
                    const long long cm = plane(k - 1) + oc;
                    const double bxn = fma(-dtdy, dEzy, fma(dtdz, eyN - eyP, pbx));
                    const double byn = fma(-dtdz, exN - exP, fma(dtdx, dEzx, pby));
                    const double bxo = COMBINE ? fma(cb.wn, qbx, cb.ws * bxn) : bxn;
                    bout[cm] = bxo;
                    if (i == 0) bout[cm + g.n[0]] = bxo;  // periodic copy: x-face n0 is face 0
                    bout[sa + cm] = COMBINE ? fma(cb.wn, qby, cb.ws * byn) : byn;
                }
                // b_z on the lower face of plane k (the last segment also writes face nz into the ghost
                // plane: see k_ct_tma)
                if (k < k1 || k1 == g.n[2]) {
                    const double eyx = sE[buf][2][ty][tx + 1], exy = sE[buf][1][ty + 1][tx];
                    const double bzn = fma(-dtdx, eyx - eyN, fma(dtdy, exy - exN, pbz));
                    bout[2 * sa + c] = COMBINE ? fma(cb.wn, qbz, cb.ws * bzn) : bzn;
                }
                if (k < k1) {
                    if (dbg) { dbg[c] = exN; dbg[sa + c] = eyN; dbg[2 * sa + c] = ez; }
                    // operands of the next iteration: b_x, b_y of this plane, b_z of the next
                    pbx = bin[c]; pby = bin[sa + c];
                    if (COMBINE) { qbx = cb.Sn[c]; qby = cb.Sn[sa + c]; }
                    if (k + 1 < k1 || k1 == g.n[2]) {
                        pbz = bin[2 * sa + c + st2];
                        if (COMBINE) qbz = cb.Sn[2 * sa + c + st2];
                    }
                }
                dEzx = ezx - ez; dEzy = ezy - ez;
            }
        }
        exP = exN; eyP = eyN;
    }
}

// ---------------------------------------------------------------- API layout <-> padded layout
// The caller's interior-only array (extent m0 x m1 x ..., planes counted from the first plane this
// process holds) <-> the padded array of one slab; kofs = the slab's first plane in the caller's array.
__global__ void k_unpack(Grid g, Box box, const double *__restrict__ src, int m0, int m1, int kofs, double *__restrict__ dst)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    dst[g.at(i, j, k)] = src[((long long)(k + kofs) * m1 + j) * m0 + i];
}

// sk0 >= 0: every plane of the box is read from plane sk0 of src (the duplicate upper z face of the
// box comes from plane 0 of the slab above / of the periodic image)
__global__ void k_pack(Grid g, Box box, const double *__restrict__ src, int m0, int m1, int kofs, int sk0, double *__restrict__ dst)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    // periodic wrap in x and y: the duplicate upper face (index n) is face 0
    int ii = i % g.n[0], jj = j % g.n[1];
    dst[((long long)(k + kofs) * m1 + j) * m0 + i] = src[g.at(ii, jj, sk0 >= 0 ? sk0 : k)];
}

// cell-centred B of the API's U[4..6]: the mean of the two faces (R7); 2D: U[6] is the stored B_z.
// bz_up: the b_z array whose plane 0 is the upper face of this slab's last plane (the slab above; the
// array itself in a periodic single domain).  n = zones of the caller's array, kofs as above.
__global__ void k_pack_cellb(Grid g, Box box, const double *__restrict__ b, const double *__restrict__ bz_up,
                             double *__restrict__ dst, long long n, int kofs)
{
    int i, j, k;
    if (!thread_zone(box, i, j, k)) return;
    const long long sa = g.sa, c = g.at(i, j, k);
    const long long o = ((long long)(k + kofs) * g.n[1] + j) * g.n[0] + i;
    dst[o] = 0.5 * (b[c] + b[g.at(wrap_p1(i, g.n[0]), j, k)]);
    dst[n + o] = 0.5 * (b[sa + c] + b[sa + g.at(i, wrap_p1(j, g.n[1]), k)]);
    if (!g.act[2]) dst[2 * n + o] = b[2 * sa + c];
    else dst[2 * n + o] = 0.5 * (b[2 * sa + c] + (k + 1 < g.n[2] ? b[2 * sa + c + g.st[2]] : bz_up[g.at(i, j, 0)]));
}

} // namespace pluto
