// ct_tma.cuh -- constrained transport (a6, R6) [+ RK2 combine of the faces (a7)] with the CT work
// arrays staged into shared memory by TMA (cp.async.bulk.tensor + mbarrier), sm_100a.
//
//   k_ct_halo : one periodic layer (i = -1, n and j = -1, n) of the twelve CT arrays, so that every
//               TMA box of k_ct_tma lies on valid data (TMA cannot wrap; out-of-array reads are zero
//               filled and never used)
//   k_ct_tma  : the CT step proper
#pragma once
#include <cuda.h>
#include "kernels.cuh"

namespace pluto {

// box of a 4D tensor (x, y, z, array) -> shared memory, completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, int c0, int c1, int c2, int c3, void *bar)
{
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes"
                 " [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------- periodic halo rows of the CT arrays
// Rows j = -1 and j = n1 of every plane the CT kernel reads (3D: -1 .. nz) receive the rows n1-1 and 0
// (positions i = -1 .. n0: the sweep kernels have already written the x copies, kernels.cuh ct_xdup).
// grid.x = plane, grid.y = array; contiguous row copies.
__global__ void __launch_bounds__(256) k_ct_halo(Grid g, double *__restrict__ ct, int two_d)
{
    const int n0 = g.n[0], n1 = g.n[1];
    const int a = blockIdx.y, k = (int)blockIdx.x - (two_d ? 0 : 1);
    if (two_d && !(a == 0 || a == 3 || a == 6 || a == 7 || a == 11)) return;     // arrays the 2D path reads
    double *arr = ct + (long long)a * g.sa + (long long)(k + g.off[2]) * g.st[2] + g.off[0] - 1;
    const long long st1 = g.st[1];
    double *lo = arr + (long long)(g.off[1] - 1) * st1, *hi = arr + (long long)(g.off[1] + n1) * st1;
    const double *s_lo = arr + (long long)(g.off[1] + n1 - 1) * st1, *s_hi = arr + (long long)g.off[1] * st1;
    for (int e = threadIdx.x; e < n0 + 2; e += blockDim.x) { lo[e] = s_lo[e]; hi[e] = s_hi[e]; }
}

// ---------------------------------------------------------------- CT with TMA-staged planes
// Block = CT_TX x CT_TY columns marching along z over `seglen` planes.  One elected thread issues,
// one plane ahead, a TMA box per CT array: the tile plus the halo column i0-1 and halo row j0-1
// ([CTM_ROWS][CTM_COLS] doubles per array, double buffered, completion on an mbarrier).  All threads
// wait on the mbarrier, then every operand of the three edge EMFs is a shared-memory load at a
// constant offset.  Iteration k forms E_z(i-1/2, j-1/2, k) and, with the plane k-1 values kept in
// registers, E_x(i, j-1/2, k-1/2), E_y(i-1/2, j, k-1/2); they are exchanged through shared memory
// (double buffered: one __syncthreads per plane) and the faces b_z(k), b_x(k-1), b_y(k-1) are
// updated with  db/dt = -curl E  (COMBINE: bout <- (bout + that)/2 in place, bout = faces of S^n).
// No edge EMF ever touches HBM and every CT value is fetched from HBM once per tile.
constexpr int CTM_COLS = CT_TX + 2, CTM_ROWS = CT_TY + 1;            // box: 34 x 9 (x extent * 8 B is a multiple of 16)
constexpr int CTM_TILE = 320;                                        // doubles per array tile, padded to 128 B multiples
constexpr int CTM_BOX_BYTES = CTM_COLS * CTM_ROWS * 8;
constexpr int CTM_SMEM_BYTES = (2 * CT_COUNT * CTM_TILE + 2 * 3 * CT_TX * CT_TY) * 8 + 64;

template <bool COMBINE, bool TWO_D>
__global__ void __launch_bounds__(CT_TX * CT_TY, 3)
k_ct_tma(Grid g, const __grid_constant__ CUtensorMap tmap, const double *__restrict__ ct,
         const double *__restrict__ bin, double *bout, const StepParams *__restrict__ P, int seglen,
         double *__restrict__ dbg, Combine cb)
{
    extern __shared__ __align__(128) unsigned char ctm_raw[];
    double *vals = reinterpret_cast<double *>(ctm_raw);                    // [2][CT_COUNT][CTM_TILE]
    double *sE = vals + 2 * CT_COUNT * CTM_TILE;                           // [2][3][CT_TY][CT_TX]
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(sE + 2 * 3 * CT_TX * CT_TY);   // [2]
    const int tx = threadIdx.x, ty = threadIdx.y;
    const bool leader = tx == 0 && ty == 0;
    const int i0 = blockIdx.x * (CT_TX - 1), j0 = blockIdx.y * (CT_TY - 1);
    const int i = i0 + tx, j = j0 + ty;
    // cells i <= n0, j <= n1 supply edges (position n holds the periodic copy of cell 0, k_ct_halo);
    // faces are updated by the inner threads
    const bool edge = i <= g.n[0] && j <= g.n[1];
    const bool upd = tx < CT_TX - 1 && ty < CT_TY - 1 && i < g.n[0] && j < g.n[1];
    const int k0 = blockIdx.z * seglen, k1 = min(k0 + seglen, g.n[2]);
    const long long sa = g.sa, st1 = g.st[1], st2 = g.st[2];
    const double dtdx = P->dtdx[0], dtdy = P->dtdx[1], dtdz = P->dtdx[2];
    auto zc = [&](int k) { return k + g.off[2]; };     // padded z coordinate of plane k (no z wrap: see k_ct)
    // in-plane offset of the own cell (idle threads are clamped onto a legal address)
    const long long oc = (long long)((edge ? j : 0) + g.off[1]) * st1 + (edge ? i : 0) + g.off[0];

    // a TMA box of doubles must start on a 16-byte boundary: the box begins at the even x coordinate at or
    // below the halo column i0-1 (its 34 columns still reach i0+31) and the tile is read at that shift
    const int xs = (g.off[0] + i0 - 1) & ~1, shift = (g.off[0] + i0 - 1) - xs;
    // the CT arrays: F_x[By] 0, F_x[Bz] 1, F_y[Bz] 2, F_y[Bx] 3, F_z[Bx] 4, F_z[By] 5, w_x 6, w_y 7, w_z 8, E^c 9-11
    auto issue = [&](int buf, int k) {                                     // leader only
        void *bar = bars + buf;
        double *dst = vals + buf * CT_COUNT * CTM_TILE;
        const int c0 = xs, c1 = g.off[1] + j0 - 1, c2 = zc(k);
        if (TWO_D) {
            mbar_expect_tx(bar, 5 * CTM_BOX_BYTES);
            tma_load_4d(dst + 0 * CTM_TILE, &tmap, c0, c1, c2, 0, bar);
            tma_load_4d(dst + 3 * CTM_TILE, &tmap, c0, c1, c2, 3, bar);
            tma_load_4d(dst + 6 * CTM_TILE, &tmap, c0, c1, c2, 6, bar);
            tma_load_4d(dst + 7 * CTM_TILE, &tmap, c0, c1, c2, 7, bar);
            tma_load_4d(dst + 11 * CTM_TILE, &tmap, c0, c1, c2, 11, bar);
        } else {
            mbar_expect_tx(bar, CT_COUNT * CTM_BOX_BYTES);
#pragma unroll
            for (int a = 0; a < CT_COUNT; a++) tma_load_4d(dst + a * CTM_TILE, &tmap, c0, c1, c2, a, bar);
        }
    };
    if (leader) {
        mbar_init(bars, 1);
        mbar_init(bars + 1, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (leader) issue(k0 & 1, k0);

    // plane k-1 values that enter E_x, E_y at k - 1/2
    double fyz = 0, wyP = 0, excP = 0, excPm = 0, fxz = 0, wxP = 0, eycP = 0, eycPm = 0;
    if (!TWO_D) {
        const double *q = ct + (long long)zc(k0 - 1) * st2 + oc;
        fyz = q[2 * sa];  wyP = q[7 * sa];
        excP = q[9 * sa]; excPm = q[9 * sa - st1];
        fxz = q[1 * sa];  wxP = q[6 * sa];
        eycP = q[10 * sa]; eycPm = q[10 * sa - 1];
    }
    double exP = 0.0, eyP = 0.0, dEzx = 0.0, dEzy = 0.0;
    // faces to update next: b_z(k), b_x(k-1), b_y(k-1) (+ the S^n faces in the combine stage)
    double pbx = 0, pby = 0, pbz = 0, qbx = 0, qby = 0, qbz = 0;
    if (upd) {
        const long long c = (long long)zc(k0) * st2 + oc;
        if (TWO_D) {
            pbx = bin[c]; pby = bin[sa + c];
            if (COMBINE) { qbx = cb.Sn[c]; qby = cb.Sn[sa + c]; }
        } else {
            pbz = bin[2 * sa + c];
            if (COMBINE) qbz = cb.Sn[2 * sa + c];
        }
    }
    const int so = (ty + 1) * CTM_COLS + tx + 1 + shift;                   // own position in a tile
    constexpr int XM = -1, YM = -CTM_COLS, XYM = -CTM_COLS - 1;

    for (int k = k0; k <= (TWO_D ? k0 : k1); k++) {
        const int buf = k & 1;
        if (leader && !TWO_D && k < k1) {
            fence_proxy_async();                 // the other buffer was read (generic proxy) one iteration ago
            issue(buf ^ 1, k + 1);
        }
        mbar_wait(bars + buf, ((k - k0) >> 1) & 1);
        const double *v = vals + buf * CT_COUNT * CTM_TILE + so;
        auto S = [&](int a, int off) { return v[a * CTM_TILE + off]; };
        const double wx = S(6, 0), wy = S(7, 0);
        // E_z(i-1/2, j-1/2, k): A = x, B = y
        const double ez = edge_emf(-S(0, YM), -S(0, 0), S(3, XM), S(3, 0), S(6, YM), wx, S(7, XM), wy,
                                   S(11, XYM), S(11, YM), S(11, XM), S(11, 0));
        double exN = 0.0, eyN = 0.0;
        double *e = sE + buf * 3 * CT_TX * CT_TY + ty * CT_TX + tx;
        e[0] = ez;
        if (!TWO_D) {
            const double wz = S(8, 0);
            // E_x(i, j-1/2, k-1/2): A = y, B = z
            const double fyzN = S(2, 0), excN = S(9, 0), excNm = S(9, YM);
            exN = edge_emf(-fyz, -fyzN, S(5, YM), S(5, 0), wyP, wy, S(8, YM), wz, excPm, excP, excNm, excN);
            // E_y(i-1/2, j, k-1/2): A = z, B = x
            const double fxzN = S(1, 0), eycN = S(10, 0), eycNm = S(10, XM);
            eyN = edge_emf(-S(4, XM), -S(4, 0), fxz, fxzN, S(8, XM), wz, wxP, wx, eycPm, eycNm, eycP, eycN);
            e[CT_TX * CT_TY] = exN; e[2 * CT_TX * CT_TY] = eyN;
            fyz = fyzN; wyP = wy; excP = excN; excPm = excNm;
            fxz = fxzN; wxP = wx; eycP = eycN; eycPm = eycNm;
        }
        __syncthreads();                         // edge EMFs visible; everybody is done with buffer `buf`
        if (upd) {
            const double ezx = e[1], ezy = e[CT_TX];
            const long long c = (long long)zc(k) * st2 + oc;
            if (TWO_D) {
                const double bxn = fma(-dtdy, ezy - ez, pbx);
                const double byn = fma(dtdx, ezx - ez, pby);
                const double bxo = COMBINE ? fma(cb.wn, qbx, cb.ws * bxn) : bxn;
                bout[c] = bxo;
                if (i == 0) bout[c + g.n[0]] = bxo;       // periodic copy: x-face n0 is face 0
                bout[sa + c] = COMBINE ? fma(cb.wn, qby, cb.ws * byn) : byn;
                if (dbg) { dbg[c] = 0.0; dbg[sa + c] = 0.0; dbg[2 * sa + c] = ez; }
            } else {
                if (k > k0) {                    // b_x, b_y of plane k-1
                    const long long cm = (long long)zc(k - 1) * st2 + oc;
                    const double bxn = fma(-dtdy, dEzy, fma(dtdz, eyN - eyP, pbx));
                    const double byn = fma(-dtdz, exN - exP, fma(dtdx, dEzx, pby));
                    const double bxo = COMBINE ? fma(cb.wn, qbx, cb.ws * bxn) : bxn;
                    bout[cm] = bxo;
                    if (i == 0) bout[cm + g.n[0]] = bxo;  // periodic copy: x-face n0 is face 0
                    bout[sa + cm] = COMBINE ? fma(cb.wn, qby, cb.ws * byn) : byn;
                }
                // b_z on the lower face of plane k.  The last segment also writes face nz, into the ghost plane:
                // the same bits as face 0 of the slab above (of this domain, if periodic), so the dt kernel
                // finds the upper face of the top cells in its own array
                if (k < k1 || k1 == g.n[2]) {
                    const double eyx = e[2 * CT_TX * CT_TY + 1], exy = e[CT_TX * CT_TY + CT_TX];
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

} // namespace pluto
