// grid.h -- padded device layout shared by the CUDA translation units of libpluto_b200.so.
//
// Every field (cell variables, face fields, work arrays) is one "array" of identical padded shape
// [tot2][tot1][px] doubles, i contiguous (SoA).  An active axis a carries `ng` ghost
// layers below and ng + 1 above (the extra one holds the upper face / edge), so cell index i in
// [-ng, n+ng) and face index i in [-ng, n+ng] both fit; face index i is the LOWER face of cell i.
// The x origin is shifted by XOFF so that interior rows start on a 128-byte boundary.
#pragma once
#include <cstddef>

namespace pluto {

constexpr int XOFF = 16;   // doubles in front of interior cell i = 0 (>= ghost)
constexpr double kGlmCr = 0.18;   // GLM variant (glm.cuh, reading R20): c_r = c_p^2 / c_h, the recommendation of [43]

struct Grid {
    int n[3];          // interior extents nx, ny, nz
    int act[3];        // axis active (n > 1 and carries ghosts)
    int ng;            // ghost layers
    int off[3];        // index of interior cell 0 along each axis inside the padded array
    int tot[3];        // padded extents (tot[0] is the pitch)
    long long st[3];   // element strides: st[0] = 1, st[1] = pitch, st[2] = pitch * tot[1]
    long long sa;      // elements per array
    double dx[3];
    double idx[3];     // 1 / dx
    double gamma;
    double igm1;       // 1 / (gamma - 1)
    double cfl;
    int limiter;
    int ndim;

    __host__ __device__ long long at(int i, int j, int k) const {
        return (long long)(k + off[2]) * st[2] + (long long)(j + off[1]) * st[1] + (i + off[0]);
    }
};

// Per-step scalars that live in device memory so that a step needs no host round trip.
struct StepParams {
    double dt;                      // dt of the step being taken
    double dtdx[3];                 // dt / dx_d, one division each (Fig. 2)
    double time;                    // sum of dt since set_state
    double dt_fixed;                // imposed dt (pluto_step_fixed_dt)
    double dt_probe;                // CFL dt of the current state (pluto_get_dt before any step)
    unsigned long long smax_bits;   // running max of (|v_d| + c_f,d)/dx_d as an IEEE bit pattern
    int err;                        // sticky: unphysical zone met
    int pad;
    double glm_ch;                  // GLM variant (glm.cuh): c_h = cfl min(dx) / dt of the step being taken
    double glm_damp;                // exp(-dt c_h / c_r)
};

// Coarse grid of CFL upper bounds left by the kernel that writes the final hydro variables of a step
// (kernels.cuh "CFL pre-filter"), read by the exact reduction (dt_kernel.cu): cell (j / bj, k / bk).
struct BoundGrid {
    unsigned long long *b;      // IEEE bit patterns of non-negative doubles; nullptr: none
    int bj, bk, nbj;            // nbj cells per plane row
    double cfac;                // max(gamma (gamma - 1), 2)
};

inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }

// Fill the layout part of a Grid.  Returns false for sizes this library does not take.
inline bool make_grid(Grid &g, int nx, int ny, int nz, int ghost)
{
    if (nx < 2 || ny < 2 || nz < 1 || ghost < 2 || ghost > XOFF) return false;
    g.n[0] = nx; g.n[1] = ny; g.n[2] = nz;
    g.ng = ghost;
    for (int a = 0; a < 3; a++) {
        g.act[a] = g.n[a] > 1;
        if (g.act[a] && g.n[a] < ghost) return false;
        g.off[a] = g.act[a] ? ghost : 0;
        g.tot[a] = g.act[a] ? g.n[a] + 2 * ghost + 1 : 1;
    }
    g.off[0] = XOFF;
    g.tot[0] = (int)round_up(XOFF + nx + ghost + 1, 16);
    g.st[0] = 1; g.st[1] = g.tot[0]; g.st[2] = (long long)g.tot[0] * g.tot[1];
    g.sa = round_up(g.st[2] * g.tot[2], 16);
    g.ndim = g.act[2] ? 3 : 2;
    return true;
}

// A state is 8 contiguous arrays: the five hydro variables and the three magnetic arrays.  Faces are
// primary (R7): the cell-centred B of an active dimension is never stored, every consumer forms
// 0.5 * (lower face + upper face) itself.  In 2D the third magnetic array holds the cell-centred B_z.
enum StateVar { S_RHO = 0, S_MX = 1, S_MY = 2, S_MZ = 3, S_EN = 4, S_B = 5, S_COUNT = 8 };

// array ids inside the single allocation
enum ArrayId {
    A_SA = 0,        // 8: state S^n (and S^{n+1})
    A_SB = 8,        // 8: stage state S^1
    A_CT = 16,       // 12: CT work arrays (kernels.cuh: CT_FEM 6, CT_W 3, CT_EC 3); staging outside a step
    A_SC = 28,       // 8: stage state S^2 (SSP-RK3 only: allocated when the integrator asks for it)
    A_COUNT_RK2 = 28,
    A_COUNT = 36
};

} // namespace pluto
