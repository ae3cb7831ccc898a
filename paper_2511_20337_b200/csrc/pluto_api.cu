// pluto_api.cu -- the C-ABI of include/pluto.h: context, memory, host<->device copies, and the
// launch sequence of one Runge-Kutta step.  No CPU fallback: without a device every call fails loudly.
//
// The box is held as one or more z-slabs ("domains", section 3.4): a periodic single
// domain is the special case of one slab that is its own neighbour.  Every kernel works on one slab; the
// only places where slabs meet are the ghost fill (z-ghost planes are pulled out of the neighbour slab's
// interior, in this process or peer-mapped from another GPU) and the single max that fixes dt.
#include "../../include/pluto.h"
#include "../../include/pluto_debug.h"
#include "kernels.cuh"
#include "ct_tma.cuh"
#include "glm.cuh"
#include "uct.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <type_traits>
#include <vector>

namespace pluto {
void launch_dtmax(const Grid &g, const double *U, StepParams *P, BoundGrid bg, int cell_b, int nblocks, cudaStream_t s);
void launch_dtfinish(const Grid &g, StepParams *P, int mode, cudaStream_t s);
void launch_advance_time(StepParams *P, cudaStream_t s);
double probe_fp64_gflops(cudaStream_t s);
}

using namespace pluto;

namespace {

enum KernelId { K_GHOST = 0, K_FLUX_XY, K_FLUX_X, K_FLUX_Y, K_FLUX_Z, K_CT, K_DTMAX, K_SCALAR, K_PACK, K_CT_HALO, K_COUNT };
const char *const kKernelNames[K_COUNT] = { "ghost_fill", "sweep_xy", "sweep_x", "sweep_y", "sweep_z", "ct",
                                            "dt_max", "scalars", "pack_unpack", "ct_halo" };

// where a neighbour slab's arrays live (this process or a peer-mapped allocation)
struct Peer {
    double *base = nullptr;     // array 0 of the neighbour's allocation (same array order)
    double *sc = nullptr;       // its S^2 arrays (RK3), if it keeps them outside `base`
    long long sa = 0;
    int n2 = 0;
    void *ipc_mapping = nullptr;    // cudaIpcOpenMemHandle result to close, if any
    unsigned char ipc_handle[64] = {};
};

struct Domain {
    Grid g{};
    int kz0 = 0;                     // first plane of the slab inside this process's part of the box
    double *base = nullptr;          // A_COUNT_RK2 (or A_COUNT) arrays, then the scalars / bound grid of slab 0
    double *sc = nullptr;            // S^2 (8 arrays) when it was allocated after pluto_init
    bool own_mem = false, own_sc = false;
    double *uct = nullptr;           // UCT-HLLD mode: the six work arrays beyond the twelve CT arrays (allocated on first use)
    int narrays = A_COUNT_RK2;
    unsigned long long *bound = nullptr;     // dt bound grid: n1 * n2 cells at most
    CUtensorMap ct_map{};
    Peer nb[2];                      // [0] the slab below, [1] the slab above
};

struct Context {
    bool init = false;
    bool have_state = false;
    bool stepped = false;
    std::vector<Domain> dom;
    int nslab = 1, first = 0;        // slabs of the whole box / first slab held here
    int nzg = 1;                     // planes of the whole box
    int nzloc = 1;                   // planes this process holds
    StepParams *P = nullptr;         // device scalars (inside slab 0's allocation), shared by the slabs here
    void *ws = nullptr;              // registered workspace
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;   // stream in use (the caller's, or own_stream)
    cudaStream_t own_stream = nullptr;
    int own_stream_dev = -1;
    long long launches = 0;
    long long captures = 0;          // whole-step graph captures since load (pluto_graph_captures)
    long long per_step[2] = { 0, 0 };
    int use_graph = 1;
    int fuse_xy = 1;
    int ct_tma = 1;
    int rk_order = 2;                // 2: SSP-RK2 (R3), 3: SSP-RK3 (Eq. 5)
    int emf = 0;                     // PLUTO_OPT_EMF: 0 contact-mode upwinding (R6), 1 UCT-HLLD (R19)
    int divb = 0;                    // PLUTO_OPT_DIVB of the next pluto_init: 0 constrained transport, 1 GLM cleaning
    bool glm = false;                // the live context runs the GLM variant (glm.cuh)
    cudaGraphExec_t graph[2] = { nullptr, nullptr };   // [0] CFL dt step, [1] fixed dt step (of the current rk_order)
    int sm_count = 148;
    char err[512] = "";
    // per-kernel CUDA-event timing (pluto_profile)
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_ev;    // pairs (start, stop)
    std::vector<int> prof_kid;
    size_t prof_used = 0;
    double prof_ms[K_COUNT] = {};
    long long prof_cnt[K_COUNT] = {};
    bool whole() const { return (int)dom.size() == nslab; }     // every slab of the box is in this process
};

Context C;

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(C.err, sizeof C.err, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(x)                                                                              \
    do {                                                                                         \
        cudaError_t e_ = (x);                                                                    \
        if (e_ != cudaSuccess) return fail(PLUTO_ECUDA, "%s: %s", #x, cudaGetErrorString(e_));   \
    } while (0)

void prof_flush()
{
    if (!C.prof_used) return;
    cudaStreamSynchronize(C.stream);
    for (size_t n = 0; n < C.prof_used; n++) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, C.prof_ev[2 * n], C.prof_ev[2 * n + 1]) == cudaSuccess) {
            C.prof_ms[C.prof_kid[n]] += ms;
            C.prof_cnt[C.prof_kid[n]] += 1;
        }
    }
    C.prof_used = 0;
}

// bracket one launch: counts it and, in profile mode, records an event pair on the launching stream
struct Launch {
    bool timed = false;
    size_t slot = 0;
    explicit Launch(int kid)
    {
        C.launches += 1;
        if (!C.prof_on) return;
        if (2 * (C.prof_used + 1) > C.prof_ev.size()) prof_flush();
        slot = C.prof_used++;
        C.prof_kid[slot] = kid;
        cudaEventRecord(C.prof_ev[2 * slot], C.stream);
        timed = true;
    }
    ~Launch() { if (timed) cudaEventRecord(C.prof_ev[2 * slot + 1], C.stream); }
};
#define LAUNCH(kid, ...) do { Launch l_(kid); __VA_ARGS__; } while (0)

double *arr(const Domain &d, int id)
{
    if (id >= A_SC && d.sc) return d.sc + (long long)(id - A_SC) * d.g.sa;
    return d.base + (long long)id * d.g.sa;
}

// the same array of a neighbour slab
double *peer_arr(const Peer &p, int id)
{
    if (id >= A_SC && p.sc) return p.sc + (long long)(id - A_SC) * p.sa;
    return p.base + (long long)id * p.sa;
}

ZSrc zsrc(const Domain &d, int state)
{
    ZSrc z;
    z.lo = peer_arr(d.nb[0], state); z.hi = peer_arr(d.nb[1], state);
    z.lo_sa = d.nb[0].sa; z.hi_sa = d.nb[1].sa;
    z.lo_n2 = d.nb[0].n2; z.hi_n2 = d.nb[1].n2;
    return z;
}

size_t bound_cells(const Grid &g) { return (size_t)g.n[1] * g.n[2]; }

// bytes of one slab: the arrays, then 256 bytes of scalars and the dt bound grid
size_t layout_bytes(const Grid &g, int narrays)
{
    return (size_t)narrays * g.sa * sizeof(double) + 256 + round_up((long long)bound_cells(g) * 8, 256);
}

dim3 grid_for(const Box &b, int bx = 128)
{
    return dim3((b.hi[0] - b.lo[0] + bx - 1) / bx, b.hi[1] - b.lo[1], b.hi[2] - b.lo[2]);
}

// index box: per axis [lo, hi) if active, else [0, 1)
Box make_box(const Grid &g, int lo0, int hi0, int lo1, int hi1, int lo2, int hi2)
{
    Box b;
    int lo[3] = { lo0, lo1, lo2 }, hi[3] = { hi0, hi1, hi2 };
    for (int a = 0; a < 3; a++) {
        b.lo[a] = g.act[a] ? lo[a] : 0;
        b.hi[a] = g.act[a] ? hi[a] : 1;
    }
    return b;
}

Box interior(const Grid &g) { return make_box(g, 0, g.n[0], 0, g.n[1], 0, g.n[2]); }

void destroy_graphs()
{
    for (auto &gr : C.graph)
        if (gr) { cudaGraphExecDestroy(gr); gr = nullptr; }
}

// planes of slab s when nz planes are cut into nslab slabs (the first nz % nslab slabs get one more)
void slab_range(int nz, int nslab, int s, int &k0, int &n)
{
    const int q = nz / nslab, r = nz % nslab;
    n = q + (s < r ? 1 : 0);
    k0 = s * q + (s < r ? s : r);
}

// TMA descriptor of the CT work arrays: dims (pitch, tot1, tot2, CT_COUNT) doubles, box = one tile of
// one array.  cuTensorMapEncodeTiled is taken from the driver through the runtime (no -lcuda).
int make_ct_map(Domain &d)
{
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                 const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn)
            return fail(PLUTO_ECUDA, "cuTensorMapEncodeTiled not available from the driver");
        encode = (EncodeFn)fn;
    }
    const Grid &g = d.g;
    cuuint64_t dims[4] = { (cuuint64_t)g.tot[0], (cuuint64_t)g.tot[1], (cuuint64_t)g.tot[2], (cuuint64_t)CT_COUNT };
    cuuint64_t strides[3] = { (cuuint64_t)g.st[1] * 8, (cuuint64_t)g.st[2] * 8, (cuuint64_t)g.sa * 8 };
    cuuint32_t box[4] = { CTM_COLS, CTM_ROWS, 1, 1 }, estr[4] = { 1, 1, 1, 1 };
    CUresult r = encode(&d.ct_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, arr(d, A_CT), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(PLUTO_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return PLUTO_OK;
}

// ---------------------------------------------------------------- launch sequences

// The fused x+y sweep spans a whole periodic row when nx is one of the instantiated block widths (every multiple of
// 32 from 64 to 256, and 512; wider rows do not fit the registers of one block): no kernel then reads an x ghost
// other than the x-face n0 (kept equal to face 0 by the CT kernel).
bool row_wraps(int nx) { return (nx % 32 == 0 && nx >= 64 && nx <= 256) || nx == 512; }

// ghost layers of the 8 arrays of one state of one slab, one launch (z planes from the neighbour slabs)
void fill_ghosts(const Domain &d, int state, bool all = false)
{
    const Grid &g = d.g;
    const ZSrc zs = zsrc(d, state);
    // only the chunked form of the fused x+y sweep reads x ghosts (k_sweep_x reads periodic images, the row-wide
    // x+y sweep wraps inside shared memory, the marching kernels stay inside the row)
    const bool chunked_xy = C.fuse_xy && g.limiter != 2 && !row_wraps(g.n[0]);
    if (!all && !chunked_xy && C.emf != 1) {      // (the UCT-HLLD edge kernel reconstructs the face fields across x too)
        const int ngh = 2 * g.ng + 1;
        const int rows = (g.act[2] ? ngh * (g.n[1] + ngh) : 0) + g.n[2] * ngh;
        LAUNCH(K_GHOST, k_ghost_yz<<<dim3(rows, S_COUNT), 128, 0, C.stream>>>(g, arr(d, state), zs));
    } else {
        LAUNCH(K_GHOST, k_ghost<<<C.sm_count * 8, 256, 0, C.stream>>>(g, arr(d, state), S_COUNT, zs));
    }
}

// segments of a marching kernel: enough independent threads for ~8 waves of 16 warps per SM,
// segments no shorter than 16 cells -- or 4 cells when the grid is so small that 16-cell segments would
// leave most SMs idle (configs 0 and 1: the step is then bound by the length of one segment's march)
int march_seglen(int n, long long columns)
{
    const long long want = (long long)C.sm_count * 16 * 32 * 8;
    long long nseg = (want + columns - 1) / columns;
    if (nseg < 1) nseg = 1;
    // equal segments when a slightly smaller count divides n (measured 2% faster at 256^3: 8 x 32 vs 10 x 26)
    for (long long m = nseg; m >= 1 && 4 * m >= 3 * nseg; m--)
        if (n % m == 0) { nseg = m; break; }
    int len = (int)((n + nseg - 1) / nseg);
    const int minlen = columns * ((n + 15) / 16) < (long long)C.sm_count * 512 ? 4 : 16;
    if (len < minlen) len = minlen;
    if (len > n) len = n;
    return len;
}

// In 3D the z sweep writes the final hydro variables of a stage; in the last stage of a step it also fills
// the dt bound grid (kernels.cuh SigmaBound).
BoundGrid bound_grid(const Domain &d, bool last, int bj, int bk)
{
    BoundGrid bg;
    bg.b = last ? d.bound : nullptr;
    bg.bj = bj; bg.bk = bk; bg.nbj = (d.g.n[1] + bj - 1) / bj;
    bg.cfac = fmax(d.g.gamma * (d.g.gamma - 1.0), 2.0);
    return bg;
}

// segment lengths of the marching sweeps (functions of the slab alone: the dt kernel must find the bound
// grid in the shape the last stage of the previous step wrote it, whatever path wrote it)
int seglen_y(const Grid &g) { return march_seglen(g.n[1], (long long)g.n[0] * g.n[2]); }
int seglen_z(const Grid &g) { return march_seglen(g.n[2], (long long)g.n[0] * g.n[1]); }

// the bound grid of the slab: one cell per (row, z segment); 2D runs keep none (the dt kernel reads every row)
BoundGrid final_bound_grid(const Domain &d, bool last)
{
    return bound_grid(d, last && d.g.act[2], 1, d.g.act[2] ? seglen_z(d.g) : 1);
}

// UCT-HLLD work arrays of a slab: the twelve CT arrays first, then the six of d.uct
UctArrays uct_arrays(const Domain &d)
{
    UctArrays A;
    for (int n = 0; n < UCT_COUNT; n++)
        A.p[n] = n < CT_COUNT ? arr(d, A_CT + n) : d.uct + (long long)(n - CT_COUNT) * d.g.sa;
    return A;
}

UctOut uct_out(const Domain &d, int dir)
{
    UctOut o;
    const UctArrays A = uct_arrays(d);
    for (int m = 0; m < 5; m++) o.p[m] = A.p[dir * 5 + m];
    return o;
}

template <int LIM, bool TWO_D, bool UCT>
void launch_sweeps(const Domain &d, const double *Sin, double *Sout, Combine cb, bool last)
{
    const Grid &g = d.g;
    cudaStream_t s = C.stream;
    double *ct = arr(d, A_CT);
    const double scale = cb.Sn ? cb.ws : 1.0;
    // 3D: the x and y sweeps cover hz planes beyond the slab on each side (the CT step reads their face data there:
    // one plane for the contact-mode rule, the reach of the transverse reconstruction for UCT-HLLD)
    const int hz = TWO_D ? 0 : (UCT ? sx_halo(LIM) : 1);
    const int kz0 = -hz;
    const int nplanes = g.n[2] + 2 * hz;
    UctOut ux{}, uy{}, uz{};
    if constexpr (UCT) { ux = uct_out(d, 0); uy = uct_out(d, 1); uz = uct_out(d, 2); }
    const BoundGrid none = bound_grid(d, false, 1, 1);
    bool fused = false;
    // In a plain Euler stage of a 3D run the z sweep goes FIRST and writes S - dt/dz dFz; the fused x+y
    // sweep then finishes the zones from there.  The read-modify-write of S' (5 + 5 doubles per zone) thereby
    // moves from the HBM-bound z sweep to the ALU-bound x+y sweep.  Combine stages keep the x+y sweep first
    // (S^n has to be read either way, and the last writer of the step fills the dt bound grid: the z sweep).
    bool zfirst = false;
    if constexpr (LIM != 2 && !TWO_D) zfirst = C.fuse_xy && !cb.Sn;
    auto z_sweep = [&](const double *base) {
        const int bx = (g.n[0] + MARCH_NT - 1) / MARCH_NT;
        const int len = seglen_z(g);
        dim3 grid(bx, g.n[1], (g.n[2] + len - 1) / len);
        const BoundGrid bg = final_bound_grid(d, last);
        if constexpr (LIM == 2) {
            if (last) LAUNCH(K_FLUX_Z, k_sweep_march_wz<2, TWO_D, !TWO_D, UCT><<<grid, MARCH_NT, WZ_SMEM_BYTES, s>>>(g, Sin, Sout, ct, C.P, scale, len, 0, bg, uz));
            else      LAUNCH(K_FLUX_Z, k_sweep_march_wz<2, TWO_D, false, UCT><<<grid, MARCH_NT, WZ_SMEM_BYTES, s>>>(g, Sin, Sout, ct, C.P, scale, len, 0, bg, uz));
        } else {
            if (last) LAUNCH(K_FLUX_Z, k_sweep_march<2, LIM, TWO_D, !TWO_D, UCT><<<grid, MARCH_NT, 0, s>>>(g, Sin, Sout, base, ct, C.P, scale, len, 0, bg, uz));
            else      LAUNCH(K_FLUX_Z, k_sweep_march<2, LIM, TWO_D, false, UCT><<<grid, MARCH_NT, 0, s>>>(g, Sin, Sout, base, ct, C.P, scale, len, 0, bg, uz));
        }
    };
    if (zfirst) z_sweep(Sin);
    if constexpr (LIM != 2) if (C.fuse_xy) {
        fused = true;
        // fused x + y sweep: one block per x-row chunk and y-segment.  The block width is a template
        // parameter (shared-memory offsets become immediates): a whole periodic row when nx is one of
        // the instantiated widths, else chunks of 128 or 256 threads that overlap by four cells.
        const int nx = g.n[0];
        const bool wrap = row_wraps(nx);
        const int nt = wrap ? nx : (nx > 124 ? 256 : 128);
        const int chunks = wrap ? 1 : (nx + nt - 5) / (nt - 4);
        const int len = seglen_y(g);
        dim3 grid(chunks, (g.n[1] + len - 1) / len, nplanes);
        const size_t smem = (size_t)XY_DOUBLES_PER_THREAD * nt * sizeof(double) + XY_SMEM_EXTRA(nt);
        void (*k)(Grid, const double *, double *, const double *, double *, StepParams *, Combine, int, int, UctOut, UctOut) =
            wrap ? (nt == 64 ? k_sweep_xy<LIM, TWO_D, true, 64, UCT> : nt == 96 ? k_sweep_xy<LIM, TWO_D, true, 96, UCT>
                    : nt == 128 ? k_sweep_xy<LIM, TWO_D, true, 128, UCT> : nt == 160 ? k_sweep_xy<LIM, TWO_D, true, 160, UCT>
                    : nt == 192 ? k_sweep_xy<LIM, TWO_D, true, 192, UCT> : nt == 224 ? k_sweep_xy<LIM, TWO_D, true, 224, UCT>
                    : nt == 256 ? k_sweep_xy<LIM, TWO_D, true, 256, UCT> : k_sweep_xy<LIM, TWO_D, true, 512, UCT>)
                 : (nt == 128 ? k_sweep_xy<LIM, TWO_D, false, 128, UCT> : k_sweep_xy<LIM, TWO_D, false, 256, UCT>);
        cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        LAUNCH(K_FLUX_XY, k<<<grid, nt, smem, s>>>(g, Sin, Sout, zfirst ? Sout : Sin, ct, C.P, cb, len, kz0, ux, uy));
    }
    if (!fused) {
        if constexpr (LIM == 2) {
            cudaFuncSetAttribute(k_sweep_march_wz<1, TWO_D, false, UCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, WZ_SMEM_BYTES);
            cudaFuncSetAttribute(k_sweep_march_wz<2, TWO_D, false, UCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, WZ_SMEM_BYTES);
            cudaFuncSetAttribute(k_sweep_march_wz<2, TWO_D, !TWO_D, UCT>, cudaFuncAttributeMaxDynamicSharedMemorySize, WZ_SMEM_BYTES);
        }
        const long long nitems = (long long)(g.n[0] + 2 * sx_halo(LIM)) * g.n[1] * nplanes;
        LAUNCH(K_FLUX_X, k_sweep_x<LIM, TWO_D, UCT><<<(unsigned)((nitems + sx_out(LIM) - 1) / sx_out(LIM)), SX_NT, 0, s>>>(
                             g, Sin, Sout, ct, C.P, cb, hz, ux));
        const int bx = (g.n[0] + MARCH_NT - 1) / MARCH_NT;
        const int len = seglen_y(g);
        dim3 grid(bx, (g.n[1] + len - 1) / len, nplanes);
        if constexpr (LIM == 2) LAUNCH(K_FLUX_Y, k_sweep_march_wz<1, TWO_D, false, UCT><<<grid, MARCH_NT, WZ_SMEM_BYTES, s>>>(g, Sin, Sout, ct, C.P, scale, len, kz0, none, uy));
        else LAUNCH(K_FLUX_Y, k_sweep_march<1, LIM, TWO_D, false, UCT><<<grid, MARCH_NT, 0, s>>>(g, Sin, Sout, Sout, ct, C.P, scale, len, kz0, none, uy));
    }
    if (!TWO_D && !zfirst) z_sweep(Sout);
}

// CT: edge EMFs + face update (+ combine) in one kernel; dbg (debug only) receives the edge EMFs
void launch_ct(const Domain &d, const double *bin, double *bout, Combine cb, double *dbg)
{
    const bool combine = cb.Sn != nullptr;
    const Grid &g = d.g;
    cudaStream_t s = C.stream;
    if (C.emf == 1) {
        // UCT-HLLD (R19, uct.cuh): halos of the face data, edge EMFs, face update
        const bool two_d = !g.act[2];
        const int h = sx_halo(g.limiter), hz = two_d ? 0 : h;
        const UctArrays A = uct_arrays(d);
        LAUNCH(K_CT_HALO, k_uct_halo<<<dim3((g.n[1] + 2 * h + UCT_HALO_ROWS - 1) / UCT_HALO_ROWS, g.n[2] + 2 * hz, UCT_FACE), 256, 0, s>>>(g, A, h, hz));
        const dim3 ge((g.n[0] + UCT_TX) / UCT_TX, (g.n[1] + UCT_TY) / UCT_TY, two_d ? 1 : g.n[2] + 1), be(UCT_TX, UCT_TY);
        if (two_d) {
            if (g.limiter == 0)      LAUNCH(K_CT, k_emf_uct<0, true><<<ge, be, 0, s>>>(g, A, bin));
            else if (g.limiter == 1) LAUNCH(K_CT, k_emf_uct<1, true><<<ge, be, 0, s>>>(g, A, bin));
            else                     LAUNCH(K_CT, k_emf_uct<2, true><<<ge, be, 0, s>>>(g, A, bin));
        } else {
            if (g.limiter == 0)      LAUNCH(K_CT, k_emf_uct<0, false><<<ge, be, 0, s>>>(g, A, bin));
            else if (g.limiter == 1) LAUNCH(K_CT, k_emf_uct<1, false><<<ge, be, 0, s>>>(g, A, bin));
            else                     LAUNCH(K_CT, k_emf_uct<2, false><<<ge, be, 0, s>>>(g, A, bin));
        }
        const dim3 gu((g.n[0] + 127) / 128, g.n[1], two_d ? 1 : g.n[2] + 1);
        if (two_d) {
            if (combine) LAUNCH(K_CT, k_ct_update<true, true><<<gu, 128, 0, s>>>(g, A, bin, bout, C.P, cb));
            else         LAUNCH(K_CT, k_ct_update<false, true><<<gu, 128, 0, s>>>(g, A, bin, bout, C.P, cb));
        } else {
            if (combine) LAUNCH(K_CT, k_ct_update<true, false><<<gu, 128, 0, s>>>(g, A, bin, bout, C.P, cb));
            else         LAUNCH(K_CT, k_ct_update<false, false><<<gu, 128, 0, s>>>(g, A, bin, bout, C.P, cb));
        }
        if (dbg) cudaMemcpyAsync(dbg, A.p[UCT_FACE], 3 * g.sa * sizeof(double), cudaMemcpyDeviceToDevice, s);
        return;
    }
    const int tiles_x = (g.n[0] + CT_TX - 2) / (CT_TX - 1), tiles_y = (g.n[1] + CT_TY - 2) / (CT_TY - 1);
    const int len = march_seglen(g.n[2], (long long)tiles_x * tiles_y * CT_TX * CT_TY);
    dim3 grid(tiles_x, tiles_y, (g.n[2] + len - 1) / len), block(CT_TX, CT_TY);
    const double *ct = arr(d, A_CT);
    if (C.ct_tma) {
        // periodic halo rows of the CT arrays (3D: planes -1 .. nz), then the TMA-staged kernel
        LAUNCH(K_CT_HALO, k_ct_halo<<<dim3(g.act[2] ? g.n[2] + 2 : 1, CT_COUNT), 256, 0, s>>>(g, arr(d, A_CT), g.act[2] ? 0 : 1));
        if (g.act[2]) {
            if (combine) LAUNCH(K_CT, k_ct_tma<true, false><<<grid, block, CTM_SMEM_BYTES, s>>>(g, d.ct_map, ct, bin, bout, C.P, len, dbg, cb));
            else         LAUNCH(K_CT, k_ct_tma<false, false><<<grid, block, CTM_SMEM_BYTES, s>>>(g, d.ct_map, ct, bin, bout, C.P, len, dbg, cb));
        } else {
            if (combine) LAUNCH(K_CT, k_ct_tma<true, true><<<grid, block, CTM_SMEM_BYTES, s>>>(g, d.ct_map, ct, bin, bout, C.P, len, dbg, cb));
            else         LAUNCH(K_CT, k_ct_tma<false, true><<<grid, block, CTM_SMEM_BYTES, s>>>(g, d.ct_map, ct, bin, bout, C.P, len, dbg, cb));
        }
        return;
    }
    const size_t smem = 0;
    if (g.act[2]) {
        if (combine) LAUNCH(K_CT, k_ct<true, false><<<grid, block, smem, s>>>(g, ct, bin, bout, C.P, len, dbg, cb));
        else         LAUNCH(K_CT, k_ct<false, false><<<grid, block, smem, s>>>(g, ct, bin, bout, C.P, len, dbg, cb));
    } else {
        if (combine) LAUNCH(K_CT, k_ct<true, true><<<grid, block, smem, s>>>(g, ct, bin, bout, C.P, len, dbg, cb));
        else         LAUNCH(K_CT, k_ct<false, true><<<grid, block, smem, s>>>(g, ct, bin, bout, C.P, len, dbg, cb));
    }
}

// The dynamic shared memory of the TMA-staged CT kernel is above the 48 KB default: the attribute is
// per device and per function, set at every pluto_init (the current device may have changed).
int set_kernel_attributes()
{
    CUDA_TRY(cudaFuncSetAttribute(k_ct_tma<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES));
    CUDA_TRY(cudaFuncSetAttribute(k_ct_tma<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES));
    CUDA_TRY(cudaFuncSetAttribute(k_ct_tma<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES));
    CUDA_TRY(cudaFuncSetAttribute(k_ct_tma<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES));
    return PLUTO_OK;
}

// One Runge-Kutta stage over the slabs held here: Sout <- Euler(Sin), or with a combine
// Sout <- wn * S^n + ws * Euler(Sin) (sn < 0: no combine; sn may equal out: in place).  Every slab's
// ghost fill comes first: it reads the neighbours' interiors of `in`, which the compute kernels of this
// stage never write (out != in).
// ---- the GLM variant (glm.cuh): cell-centred B in the three magnetic arrays of a state, psi and the scratch
// state of the combine stages in the (otherwise unused) CT work arrays
int glm_psi(int state) { return A_CT + (state == A_SA ? 0 : state == A_SB ? 1 : 2); }
constexpr int GLM_TMP = A_CT + 3, GLM_TMP_PSI = A_CT + 11;

template <int LIM>
void enqueue_stage_glm(int in, int out, int sn, double wn, double ws, bool last)
{
    const Domain &d = C.dom[0];
    const Grid &g = d.g;
    cudaStream_t s = C.stream;
    ZSrc zs = zsrc(d, in);
    LAUNCH(K_GHOST, k_ghost<<<C.sm_count * 8, 256, 0, s>>>(g, arr(d, in), S_COUNT, zs));
    double *psin = arr(d, glm_psi(in));
    ZSrc zp = zs;
    zp.lo = zp.hi = psin;
    LAUNCH(K_GHOST, k_ghost<<<C.sm_count * 2, 256, 0, s>>>(g, psin, 1, zp));
    // a combine stage computes Euler(S) into scratch arrays first (out may be S^n itself)
    double *So = arr(d, sn >= 0 ? GLM_TMP : out), *po = arr(d, sn >= 0 ? GLM_TMP_PSI : glm_psi(out));
    const dim3 grid((g.n[0] + 127) / 128, g.n[1], g.n[2]);
    const dim3 gx((g.n[0] + GLMX_NT - 5) / (GLMX_NT - 4), g.n[1], g.n[2]);
    LAUNCH(K_FLUX_X, k_glm_sweep_x<LIM, true><<<gx, GLMX_NT, 0, s>>>(g, arr(d, in), psin, So, po, C.P));
    // the last sweep of a combine stage writes wn * S^n + ws * Euler(S) (and damps psi at the end of a step) itself;
    // the z march of the last stage also leaves the dt bound grid
    const bool comb = sn >= 0, three_d = g.act[2] != 0;
    GlmCombine cg{};
    if (comb) cg = GlmCombine{ arr(d, out), arr(d, glm_psi(out)), arr(d, sn), arr(d, glm_psi(sn)), wn, ws, last ? 1 : 0 };
    const BoundGrid none = bound_grid(d, false, 1, 1);
    {
        const int len = seglen_y(g);
        const dim3 gy((g.n[0] + 127) / 128, (g.n[1] + len - 1) / len, g.n[2]);
        if (comb && !three_d) LAUNCH(K_FLUX_Y, k_glm_march<1, LIM, false, true, false><<<gy, 128, 0, s>>>(g, arr(d, in), psin, So, po, C.P, len, cg, none));
        else                  LAUNCH(K_FLUX_Y, k_glm_march<1, LIM, false, false, false><<<gy, 128, 0, s>>>(g, arr(d, in), psin, So, po, C.P, len, cg, none));
    }
    if (three_d) {
        const int len = seglen_z(g);
        const dim3 gz((g.n[0] + 127) / 128, g.n[1], (g.n[2] + len - 1) / len);
        const BoundGrid bg = final_bound_grid(d, last);
        if (comb && last) LAUNCH(K_FLUX_Z, k_glm_march<2, LIM, false, true, true><<<gz, 128, 0, s>>>(g, arr(d, in), psin, So, po, C.P, len, cg, bg));
        else if (comb)    LAUNCH(K_FLUX_Z, k_glm_march<2, LIM, false, true, false><<<gz, 128, 0, s>>>(g, arr(d, in), psin, So, po, C.P, len, cg, none));
        else              LAUNCH(K_FLUX_Z, k_glm_march<2, LIM, false, false, false><<<gz, 128, 0, s>>>(g, arr(d, in), psin, So, po, C.P, len, cg, none));
    }
}

void enqueue_stage(int in, int out, int sn, double wn, double ws, bool last, double *dbg = nullptr)
{
    if (C.glm) {
        if (C.dom[0].g.limiter == 0) enqueue_stage_glm<0>(in, out, sn, wn, ws, last);
        else                         enqueue_stage_glm<1>(in, out, sn, wn, ws, last);
        return;
    }
    for (const Domain &d : C.dom) fill_ghosts(d, in);
    for (const Domain &d : C.dom) {
        const Grid &g = d.g;
        const bool two_d = !g.act[2];
        const Combine cb = { sn >= 0 ? arr(d, sn) : nullptr, wn, ws };
        auto sweeps = [&](auto lim, auto twod) {
            constexpr int L = decltype(lim)::value;
            constexpr bool T = decltype(twod)::value;
            if (C.emf == 1) launch_sweeps<L, T, true>(d, arr(d, in), arr(d, out), cb, last);
            else            launch_sweeps<L, T, false>(d, arr(d, in), arr(d, out), cb, last);
        };
        using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>; using I2 = std::integral_constant<int, 2>;
        if (g.limiter == 0)      { if (two_d) sweeps(I0{}, std::true_type{}); else sweeps(I0{}, std::false_type{}); }
        else if (g.limiter == 1) { if (two_d) sweeps(I1{}, std::true_type{}); else sweeps(I1{}, std::false_type{}); }
        else                     { if (two_d) sweeps(I2{}, std::true_type{}); else sweeps(I2{}, std::false_type{}); }
        const Combine cbf = { sn >= 0 ? arr(d, sn + S_B) : nullptr, wn, ws };
        launch_ct(d, arr(d, in + S_B), arr(d, out + S_B), cbf, dbg);
    }
}

// stage s of the step (0-based); SSP-RK2 (R3) or SSP-RK3 (Eq. 5; R17: the last stage carries 2 L**)
void enqueue_rk_stage(int s)
{
    if (C.rk_order == 3) {
        if (s == 0) enqueue_stage(A_SA, A_SB, -1, 0.0, 1.0, false);                    // S*   = S^n + L(S^n)
        if (s == 1) enqueue_stage(A_SB, A_SC, A_SA, 0.75, 0.25, false);                // S**  = (3 S^n + S* + L(S*)) / 4
        if (s == 2) enqueue_stage(A_SC, A_SA, A_SA, 1.0 / 3.0, 2.0 / 3.0, true);       // S^{n+1} = (S^n + 2 (S** + L(S**))) / 3
    } else {
        if (s == 0) enqueue_stage(A_SA, A_SB, -1, 0.0, 1.0, false);                    // S^1 = S^n + L(S^n)
        if (s == 1) enqueue_stage(A_SB, A_SA, A_SA, 0.5, 0.5, true);                   // S^{n+1} = (S^n + S^1 + L(S^1)) / 2
    }
}

// exact max of the CFL candidates over the slabs held here (into P->smax_bits); the bound grid is spent
void enqueue_dtmax(bool keep_bounds)
{
    for (const Domain &d : C.dom) {
        BoundGrid bg = final_bound_grid(d, true);
        LAUNCH(K_DTMAX, launch_dtmax(d.g, arr(d, A_SA), C.P, bg, C.glm ? 1 : 0, C.sm_count * 8, C.stream));
    }
    if (!keep_bounds)
        for (const Domain &d : C.dom) cudaMemsetAsync(d.bound, 0, bound_cells(d.g) * 8, C.stream);
}

// no bound known for the current state: every row is visited
void reset_bounds()
{
    for (const Domain &d : C.dom) cudaMemsetAsync(d.bound, 0x7f, bound_cells(d.g) * 8, C.stream);
}

void enqueue_dt(int mode)
{
    if (mode != 1) enqueue_dtmax(mode == 2);
    LAUNCH(K_SCALAR, launch_dtfinish(C.dom[0].g, C.P, mode, C.stream));
}

void enqueue_step(bool fixed)
{
    enqueue_dt(fixed ? 1 : 0);
    for (int s = 0; s < C.rk_order; s++) enqueue_rk_stage(s);
    LAUNCH(K_SCALAR, launch_advance_time(C.P, C.stream));
}

int ensure_rk3_storage();
int ensure_uct_storage();

int run_steps(int nsteps, bool fixed)
{
    if (!C.whole()) return fail(PLUTO_ESTATE, "this process holds %d of %d slabs: drive the step with pluto_step_begin / pluto_step_stage",
                                (int)C.dom.size(), C.nslab);
    if (int rc = ensure_rk3_storage()) return rc;
    if (int rc = ensure_uct_storage()) return rc;
    const int gi = fixed ? 1 : 0;
    const bool graph = C.use_graph && !C.prof_on;
    if (graph && !C.graph[gi] && nsteps > 0) {
        long long before = C.launches;
        cudaGraph_t graph = nullptr;
        CUDA_TRY(cudaStreamBeginCapture(C.stream, cudaStreamCaptureModeThreadLocal));
        enqueue_step(fixed);
        cudaError_t e = cudaStreamEndCapture(C.stream, &graph);
        if (e != cudaSuccess) return fail(PLUTO_ECUDA, "graph capture: %s", cudaGetErrorString(e));
        e = cudaGraphInstantiate(&C.graph[gi], graph, 0);
        cudaGraphDestroy(graph);
        if (e != cudaSuccess) return fail(PLUTO_ECUDA, "graph instantiate: %s", cudaGetErrorString(e));
        C.captures++;
        C.per_step[gi] = C.launches - before;
        C.launches = before;                      // capture enqueued nothing
    }
    for (int s = 0; s < nsteps; s++) {
        if (graph) {
            CUDA_TRY(cudaGraphLaunch(C.graph[gi], C.stream));
            C.launches += C.per_step[gi];
        } else {
            enqueue_step(fixed);
        }
    }
    CUDA_TRY(cudaGetLastError());
    if (nsteps > 0) C.stepped = true;
    return PLUTO_OK;
}

int finish()
{
    CUDA_TRY(cudaStreamSynchronize(C.stream));
    int err = 0;
    CUDA_TRY(cudaMemcpy(&err, &C.P->err, sizeof(int), cudaMemcpyDeviceToHost));
    if (err) return fail(PLUTO_EPHYS, "non-finite or non-positive density/pressure met");
    return PLUTO_OK;
}

bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// extents of the caller's array for the face family d (d = -1: cell array) over nz planes
void api_extent(const Grid &g, int nz, int d, int m[3])
{
    m[0] = g.n[0] + (d == 0 ? 1 : 0);
    m[1] = g.n[1] + (d == 1 ? 1 : 0);
    m[2] = nz + (d == 2 ? 1 : 0);
}

size_t api_count(const Grid &g, int nz, int d)
{
    int m[3];
    api_extent(g, nz, d, m);
    return (size_t)m[0] * m[1] * m[2];
}

// Host-copy staging: the CT work arrays of the slabs are free outside a step.  With one slab they hold
// the whole caller's array (12 padded arrays > 11 interior arrays); with several slabs a temporary is used.
struct Staging {
    double *p = nullptr;
    bool temp = false;
    int get(size_t doubles)
    {
        const Domain &d0 = C.dom[0];
        if (C.dom.size() == 1 && !C.glm && doubles <= (size_t)CT_COUNT * d0.g.sa) { p = arr(d0, A_CT); return PLUTO_OK; }
        if (cudaMalloc((void **)&p, doubles * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            p = nullptr;
            return fail(PLUTO_ENOMEM, "cannot allocate %zu bytes of staging", doubles * sizeof(double));
        }
        temp = true;
        return PLUTO_OK;
    }
    ~Staging() { if (temp && p) cudaFree(p); }
};

void free_domains()
{
    for (Domain &d : C.dom) {
        for (Peer &p : d.nb)
            if (p.ipc_mapping) { cudaIpcCloseMemHandle(p.ipc_mapping); p.ipc_mapping = nullptr; }
        if (d.own_sc && d.sc) cudaFree(d.sc);
        if (d.uct) cudaFree(d.uct);
        if (d.own_mem && d.base) cudaFree(d.base);
    }
    C.dom.clear();
    C.P = nullptr;
}

// SSP-RK3 keeps a third state: allocated on first use when pluto_init ran with the RK2 layout
int ensure_rk3_storage()
{
    if (C.rk_order != 3) return PLUTO_OK;
    bool changed = false;            // captured graphs hold the S^2 pointers: they are stale only if one moved
    for (Domain &d : C.dom) {
        if (d.narrays >= A_COUNT || d.sc) continue;
        if (!C.whole()) return fail(PLUTO_ESTATE, "select SSP-RK3 before pluto_init_slabs (peers map one allocation per slab)");
        const size_t bytes = (size_t)S_COUNT * d.g.sa * sizeof(double);
        cudaError_t e = cudaMalloc((void **)&d.sc, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); d.sc = nullptr; return fail(PLUTO_ENOMEM, "cudaMalloc(%zu) for the RK3 stage state: %s", bytes, cudaGetErrorString(e)); }
        d.own_sc = true;
        changed = true;
        CUDA_TRY(cudaMemsetAsync(d.sc, 0, bytes, C.stream));
    }
    // neighbours inside this process: their S^2 lives where arr() finds it
    for (size_t s = 0; s < C.dom.size(); s++) {
        Domain &d = C.dom[s];
        if (C.whole()) {
            double *lo = C.dom[(s + C.dom.size() - 1) % C.dom.size()].sc;
            double *hi = C.dom[(s + 1) % C.dom.size()].sc;
            if (d.nb[0].sc != lo || d.nb[1].sc != hi) changed = true;
            d.nb[0].sc = lo;
            d.nb[1].sc = hi;
        }
    }
    if (changed) destroy_graphs();
    return PLUTO_OK;
}

// UCT-HLLD mode needs 18 work arrays (15 of face data, 3 edge EMFs): the twelve CT arrays and six more
int ensure_uct_storage()
{
    if (C.emf != 1 || C.glm) return PLUTO_OK;
    for (Domain &d : C.dom) {
        if (d.uct) continue;
        const size_t bytes = (size_t)(UCT_COUNT - CT_COUNT) * d.g.sa * sizeof(double);
        cudaError_t e = cudaMalloc((void **)&d.uct, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); d.uct = nullptr; return fail(PLUTO_ENOMEM, "cudaMalloc(%zu) for the UCT-HLLD work arrays: %s", bytes, cudaGetErrorString(e)); }
        // NaN patterns: a kernel that used a location no kernel had written would carry a NaN into the state
        CUDA_TRY(cudaMemsetAsync(d.uct, 0xFF, bytes, C.stream));
        destroy_graphs();
    }
    return PLUTO_OK;
}

// everything pluto_finalize does, except forgetting the registered workspace (pluto_init re-creates a live context)
void release()
{
    if (C.init) {
        cudaStreamSynchronize(C.stream);
        destroy_graphs();
    }
    free_domains();
    C.init = false; C.have_state = false; C.stepped = false;
    C.nslab = 1; C.first = 0;
}

int init_common(int nslab, int first, int count, int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess) { cudaGetLastError(); ndev = 0; }
    if (ndev < 1) return fail(PLUTO_ECUDA, "no CUDA device: this library has no CPU fallback");
    // every argument is checked before the live context is touched: a call rejected with PLUTO_EINVAL (or with
    // PLUTO_ENOMEM for a registered workspace that is too small) leaves the previous context, its state and its
    // peer mappings as they were
    if (nslab < 1 || first < 0 || count < 1 || first + count > nslab) return fail(PLUTO_EINVAL, "bad slab range");
    Grid gg;
    if (!make_grid(gg, nx, ny, nz, ghost))
        return fail(PLUTO_EINVAL, "need nx >= 2, ny >= 2, nz >= 1, 2 <= ghost <= %d, active extents >= ghost", XOFF);
    if (!(gamma > 1.0) || !(cfl > 0.0) || limiter < PLUTO_MINMOD || limiter > PLUTO_WENOZ)
        return fail(PLUTO_EINVAL, "need gamma > 1, cfl > 0, limiter in {0,1,2}");
    if (limiter == PLUTO_WENOZ && ghost < 3)
        return fail(PLUTO_EINVAL, "the WENO-Z stencil needs ghost >= 3");
    if (nslab > 1 && (nz / nslab < ghost + 1))
        return fail(PLUTO_EINVAL, "every z slab needs at least ghost + 1 = %d planes", ghost + 1);
    if (C.divb == 1 && (nslab != 1 || limiter == PLUTO_WENOZ))
        return fail(PLUTO_EINVAL, "the GLM variant runs PLM on a single domain");
    const int narrays = C.rk_order == 3 ? A_COUNT : A_COUNT_RK2;
    {
        size_t need = 0;
        for (int s = 0; s < count; s++) {
            Grid gs;
            int k0 = 0, nzl = nz;
            slab_range(nz, nslab, first + s, k0, nzl);
            if (!make_grid(gs, nx, ny, nzl, ghost)) return fail(PLUTO_EINVAL, "bad slab");
            if ((long long)gs.tot[2] * 8 > 65535 || gs.tot[1] > 65535) return fail(PLUTO_EINVAL, "extent too large for the launch grid");
            need += layout_bytes(gs, narrays);
        }
        if (C.ws && C.ws_bytes < need) return fail(PLUTO_ENOMEM, "workspace has %zu bytes, need %zu", C.ws_bytes, need);
    }
    release();
    int dev = 0;
    cudaGetDevice(&dev);
    if (!C.stream || (C.stream == C.own_stream && C.own_stream_dev != dev)) {
        C.stream = nullptr;
        int rc = pluto_set_stream(nullptr);
        if (rc) return rc;
    }
    C.glm = C.divb == 1;
    C.nslab = nslab; C.first = first; C.nzg = nz;
    C.dom.resize(count);
    int kbase = 0, dummy = 0;
    slab_range(nz, nslab, first, kbase, dummy);
    size_t total = 0;
    for (int s = 0; s < count; s++) {
        Domain &d = C.dom[s];
        int k0 = 0, nzl = nz;
        slab_range(nz, nslab, first + s, k0, nzl);
        if (!make_grid(d.g, nx, ny, nzl, ghost)) { C.dom.clear(); return fail(PLUTO_EINVAL, "bad slab"); }
        if ((long long)d.g.tot[2] * 8 > 65535 || d.g.tot[1] > 65535) { C.dom.clear(); return fail(PLUTO_EINVAL, "extent too large for the launch grid"); }
        d.g.gamma = gamma; d.g.igm1 = 1.0 / (gamma - 1.0); d.g.cfl = cfl; d.g.limiter = limiter;
        for (int a = 0; a < 3; a++) { d.g.dx[a] = 1.0 / nx; d.g.idx[a] = 1.0 / d.g.dx[a]; }   // R11: Lx = 1, cubic cells
        d.kz0 = k0 - kbase;
        d.narrays = narrays;
        total += layout_bytes(d.g, narrays);
    }
    C.nzloc = C.dom.back().kz0 + C.dom.back().g.n[2];
    // memory: the registered workspace (one piece per slab, in order) or our own allocations
    if (C.ws) {
        if (C.ws_bytes < total) { C.dom.clear(); return fail(PLUTO_ENOMEM, "workspace has %zu bytes, need %zu", C.ws_bytes, total); }
        char *p = (char *)C.ws;
        for (Domain &d : C.dom) { d.base = (double *)p; d.own_mem = false; p += layout_bytes(d.g, narrays); }
    } else {
        for (Domain &d : C.dom) {
            const size_t bytes = layout_bytes(d.g, narrays);
            cudaError_t e = cudaMalloc((void **)&d.base, bytes);
            if (e != cudaSuccess) {
                cudaGetLastError();
                d.base = nullptr;
                free_domains();
                return fail(PLUTO_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e));
            }
            d.own_mem = true;
        }
    }
    cudaDeviceGetAttribute(&C.sm_count, cudaDevAttrMultiProcessorCount, dev);
    for (Domain &d : C.dom) {
        cudaError_t e = cudaMemsetAsync(d.base, 0, layout_bytes(d.g, narrays), C.stream);
        if (e != cudaSuccess) { free_domains(); return fail(PLUTO_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e)); }
        d.bound = (unsigned long long *)((char *)d.base + (size_t)narrays * d.g.sa * sizeof(double) + 256);
    }
    C.P = (StepParams *)(C.dom[0].base + (long long)narrays * C.dom[0].g.sa);
    // neighbours inside this process; the two outer ones are peers unless the whole box is here
    for (int s = 0; s < count; s++) {
        Domain &d = C.dom[s];
        for (int side = 0; side < 2; side++) {
            int t = s + (side ? 1 : -1);
            if (C.whole()) t = (t + count) % count;
            if (t < 0 || t >= count) continue;            // attached later with pluto_attach_peer
            d.nb[side].base = C.dom[t].base; d.nb[side].sa = C.dom[t].g.sa; d.nb[side].n2 = C.dom[t].g.n[2];
        }
    }
    if (cudaStreamSynchronize(C.stream) != cudaSuccess) { free_domains(); return fail(PLUTO_ECUDA, "device memset failed"); }
    int rc = set_kernel_attributes();
    for (Domain &d : C.dom) if (!rc) rc = make_ct_map(d);
    if (rc) { free_domains(); return rc; }
    C.init = true; C.have_state = false; C.stepped = false; C.launches = 0;
    return PLUTO_OK;
}

bool peers_attached()
{
    for (const Domain &d : C.dom)
        if (!d.nb[0].base || !d.nb[1].base) return false;
    return true;
}

// GLM variant: the caller's U[8] (cell-centred B in U[4..6]) and psi <-> the padded arrays.  to_device: U
// in (psi untouched unless given); otherwise out.  Host pointers go through a temporary device buffer.
int copy_state_glm(double *U, double *psi, bool to_device)
{
    const Domain &d = C.dom[0];
    const Grid &g = d.g;
    cudaStream_t s = C.stream;
    const size_t n = api_count(g, g.n[2], -1);
    Box in = interior(g);
    const int arr_of[8] = { 0, 1, 2, 3, 5, 6, 7, 4 };          // U component -> state array (E is array 4)
    Staging st;
    double *dU = U, *dpsi = psi;
    const bool uhost = U && !is_device_ptr(U), phost = psi && !is_device_ptr(psi);
    if (uhost || phost) {
        if (int rc = st.get(9 * n)) return rc;
        if (uhost) dU = st.p;
        if (phost) dpsi = st.p + 8 * n;
    }
    if (to_device) {
        if (uhost) CUDA_TRY(cudaMemcpyAsync(dU, U, 8 * n * sizeof(double), cudaMemcpyHostToDevice, s));
        if (phost) CUDA_TRY(cudaMemcpyAsync(dpsi, psi, n * sizeof(double), cudaMemcpyHostToDevice, s));
        if (U) for (int v = 0; v < 8; v++)
            k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dU + (size_t)v * n, g.n[0], g.n[1], 0, arr(d, A_SA + arr_of[v]));
        if (psi) k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dpsi, g.n[0], g.n[1], 0, arr(d, glm_psi(A_SA)));
    } else {
        if (U) for (int v = 0; v < 8; v++)
            k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_SA + arr_of[v]), g.n[0], g.n[1], 0, -1, dU + (size_t)v * n);
        if (psi) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, glm_psi(A_SA)), g.n[0], g.n[1], 0, -1, dpsi);
        if (uhost) CUDA_TRY(cudaMemcpyAsync(U, dU, 8 * n * sizeof(double), cudaMemcpyDeviceToHost, s));
        if (phost) CUDA_TRY(cudaMemcpyAsync(psi, dpsi, n * sizeof(double), cudaMemcpyDeviceToHost, s));
    }
    C.launches += (U ? 8 : 0) + (psi ? 1 : 0);
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
}

int set_state_glm(const double *U)
{
    if (!U) return fail(PLUTO_EINVAL, "null pointer");
    const Domain &d = C.dom[0];
    CUDA_TRY(cudaMemsetAsync(arr(d, glm_psi(A_SA)), 0, (size_t)d.g.sa * sizeof(double), C.stream));     // psi = 0
    if (int rc = copy_state_glm(const_cast<double *>(U), nullptr, true)) return rc;
    reset_bounds();
    StepParams p0;
    memset(&p0, 0, sizeof p0);
    CUDA_TRY(cudaMemcpyAsync(C.P, &p0, sizeof p0, cudaMemcpyHostToDevice, C.stream));
    CUDA_TRY(cudaStreamSynchronize(C.stream));
    C.have_state = true; C.stepped = false;
    return PLUTO_OK;
}

} // namespace

// error reporting for the entry points that live in other translation units (dt_kernel.cu): same buffer as
// fail(), read back with pluto_last_error
namespace pluto {
int report_error(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(C.err, sizeof C.err, fmt, ap);
    va_end(ap);
    return code;
}
}

// ================================================================== C ABI

extern "C" {

const char *pluto_last_error(void) { return C.err; }

int pluto_device_count(void)
{
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess) { cudaGetLastError(); return 0; }
    return n;
}

size_t pluto_workspace_bytes(int nx, int ny, int nz, int ghost)
{
    return pluto_workspace_bytes_slabs(1, 0, 1, nx, ny, nz, ghost, 2);
}

size_t pluto_workspace_bytes_slabs(int nslab, int first, int count, int nx, int ny, int nz, int ghost, int rk_order)
{
    if (nslab < 1 || first < 0 || count < 1 || first + count > nslab || (rk_order != 2 && rk_order != 3)) return 0;
    if (nslab > 1 && nz / nslab < ghost + 1) return 0;
    size_t total = 0;
    for (int s = first; s < first + count; s++) {
        int k0, nzl;
        slab_range(nz, nslab, s, k0, nzl);
        Grid g;
        if (!make_grid(g, nx, ny, nzl, ghost)) return 0;
        total += layout_bytes(g, rk_order == 3 ? A_COUNT : A_COUNT_RK2);
    }
    return total;
}

int pluto_set_workspace(void *dev, size_t bytes)
{
    if (C.init && !C.dom.empty() && !C.dom[0].own_mem) return fail(PLUTO_ESTATE, "workspace in use: call pluto_finalize first");
    if (dev && !is_device_ptr(dev)) return fail(PLUTO_EINVAL, "workspace is not device memory");
    if (dev && ((size_t)dev & 255)) return fail(PLUTO_EINVAL, "workspace must be 256-byte aligned");
    C.ws = dev;
    C.ws_bytes = dev ? bytes : 0;
    return PLUTO_OK;
}

int pluto_set_stream(void *cuda_stream)
{
    if (C.init) cudaStreamSynchronize(C.stream);
    if (!cuda_stream) {
        // the legacy default stream cannot be captured into a graph: use a stream of our own, on the current device
        int dev = 0;
        if (pluto_device_count() > 0) cudaGetDevice(&dev);
        if (C.own_stream && C.own_stream_dev != dev) { cudaStreamDestroy(C.own_stream); C.own_stream = nullptr; }
        if (!C.own_stream && pluto_device_count() > 0) {
            if (cudaStreamCreateWithFlags(&C.own_stream, cudaStreamNonBlocking) != cudaSuccess) {
                cudaGetLastError();
                return fail(PLUTO_ECUDA, "cannot create a stream");
            }
            C.own_stream_dev = dev;
        }
        C.stream = C.own_stream;
    } else {
        C.stream = (cudaStream_t)cuda_stream;
    }
    destroy_graphs();
    return PLUTO_OK;
}

int pluto_finalize(void)
{
    release();
    // the registration of a workspace ends here (pluto.h: the caller keeps it alive until pluto_finalize)
    C.ws = nullptr; C.ws_bytes = 0;
    return PLUTO_OK;
}

int pluto_init(int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter)
{
    return init_common(1, 0, 1, nx, ny, nz, ghost, gamma, cfl, limiter);
}

int pluto_init_slabs(int nslab, int first, int count, int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter)
{
    if (nz < 2) return fail(PLUTO_EINVAL, "the z-slab decomposition needs a 3D box");
    return init_common(nslab, first, count, nx, ny, nz, ghost, gamma, cfl, limiter);
}

int pluto_slab_planes(int nz, int nslab, int slab, int *k0, int *planes)
{
    if (nz < 1 || nslab < 1 || slab < 0 || slab >= nslab) return fail(PLUTO_EINVAL, "bad slab");
    int kb = 0, n = 0;
    slab_range(nz, nslab, slab, kb, n);
    if (k0) *k0 = kb;
    if (planes) *planes = n;
    return PLUTO_OK;
}

int pluto_local_planes(int *k0, int *nz_local)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    int kb = 0, n = 0;
    slab_range(C.nzg, C.nslab, C.first, kb, n);
    if (k0) *k0 = kb;
    if (nz_local) *nz_local = C.nzloc;
    return PLUTO_OK;
}

int pluto_export_slab(int side, void *ipc_handle64, void **device_ptr, long long *array_stride, int *planes)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (side != 0 && side != 1) return fail(PLUTO_EINVAL, "side must be 0 (lowest slab) or 1 (highest slab)");
    const Domain &d = side ? C.dom.back() : C.dom.front();
    if (ipc_handle64) {
        if (!d.own_mem) return fail(PLUTO_ESTATE, "a slab inside a registered workspace cannot be exported by IPC handle");
        cudaIpcMemHandle_t h;
        CUDA_TRY(cudaIpcGetMemHandle(&h, d.base));
        static_assert(sizeof(h) == 64, "cudaIpcMemHandle_t is 64 bytes");
        memcpy(ipc_handle64, &h, 64);
    }
    if (device_ptr) *device_ptr = d.base;
    if (array_stride) *array_stride = d.g.sa;
    if (planes) *planes = d.g.n[2];
    return PLUTO_OK;
}

int pluto_attach_peer(int side, const void *ipc_handle64, void *device_ptr, long long array_stride, int planes)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (side != 0 && side != 1) return fail(PLUTO_EINVAL, "side must be 0 (the slab below) or 1 (the slab above)");
    if (C.whole()) return fail(PLUTO_ESTATE, "every slab is in this process: there is no peer");
    if (planes < C.dom[0].g.ng + 1 || array_stride <= 0) return fail(PLUTO_EINVAL, "bad peer layout");
    Domain &d = side ? C.dom.back() : C.dom.front();
    Peer &p = d.nb[side];
    Peer &other = (side ? C.dom.front() : C.dom.back()).nb[1 - side];
    if (p.ipc_mapping) { cudaIpcCloseMemHandle(p.ipc_mapping); p.ipc_mapping = nullptr; }
    void *ptr = device_ptr;
    if (ipc_handle64) {
        if (other.ipc_mapping && !memcmp(other.ipc_handle, ipc_handle64, 64)) {
            // two processes: the slab below and the slab above are the same allocation, mapped once
            ptr = other.ipc_mapping;
            other.ipc_mapping = nullptr;          // this side closes it
        } else {
            cudaIpcMemHandle_t h;
            memcpy(&h, ipc_handle64, 64);
            CUDA_TRY(cudaIpcOpenMemHandle(&ptr, h, cudaIpcMemLazyEnablePeerAccess));
        }
        p.ipc_mapping = ptr;
        memcpy(p.ipc_handle, ipc_handle64, 64);
    }
    if (!ptr) return fail(PLUTO_EINVAL, "need an IPC handle or a device pointer");
    p.base = (double *)ptr; p.sa = array_stride; p.n2 = planes; p.sc = nullptr;
    return PLUTO_OK;
}

int pluto_set_box(double Lx, double Ly, double Lz)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (!(Lx > 0.0) || !(Ly > 0.0) || !(Lz > 0.0)) return fail(PLUTO_EINVAL, "box lengths must be positive");
    const int n[3] = { C.dom[0].g.n[0], C.dom[0].g.n[1], C.nzg };      // Lz is the length of the WHOLE box
    const double L[3] = { Lx, Ly, Lz };
    for (Domain &d : C.dom)
        for (int a = 0; a < 3; a++) { d.g.dx[a] = L[a] / n[a]; d.g.idx[a] = 1.0 / d.g.dx[a]; }
    destroy_graphs();          // kernels take the grid by value: captured copies are stale
    // the dt bound grid was built with the old 1/dx: after a change of the box the bounds left by the last step may
    // lie below the true candidates, and filter 0 of k_dtmax would then skip the row that holds the maximum
    if (C.have_state) reset_bounds();
    return PLUTO_OK;
}

int pluto_set_option(int opt, int value)
{
    if (opt == PLUTO_OPT_GRAPH) { int old = C.use_graph; C.use_graph = value ? 1 : 0; return old; }
    if (opt == PLUTO_OPT_RK_ORDER) {
        if (value != 2 && value != 3) return fail(PLUTO_EINVAL, "rk order must be 2 or 3");
        int old = C.rk_order;
        C.rk_order = value;
        destroy_graphs();
        return old;
    }
    if (opt == PLUTO_OPT_CT_TMA) {
        int old = C.ct_tma;
        C.ct_tma = value ? 1 : 0;
        destroy_graphs();
        return old;
    }
    if (opt == PLUTO_OPT_EMF) {
        if (value != PLUTO_EMF_CONTACT && value != PLUTO_EMF_UCT_HLLD) return fail(PLUTO_EINVAL, "EMF average must be PLUTO_EMF_CONTACT or PLUTO_EMF_UCT_HLLD");
        int old = C.emf;
        C.emf = value;
        destroy_graphs();
        return old;
    }
    if (opt == PLUTO_OPT_DIVB) {
        if (value != PLUTO_DIVB_CT && value != PLUTO_DIVB_GLM) return fail(PLUTO_EINVAL, "divergence control must be PLUTO_DIVB_CT or PLUTO_DIVB_GLM");
        int old = C.divb;
        C.divb = value;                          // takes effect at the next pluto_init
        return old;
    }
    if (opt == PLUTO_OPT_FUSE_XY) {
        int old = C.fuse_xy;
        C.fuse_xy = value ? 1 : 0;
        destroy_graphs();
        return old;
    }
    return fail(PLUTO_EINVAL, "unknown option %d", opt);
}

int pluto_set_state(const double *U, const double *Bface)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (C.glm) return set_state_glm(U);
    if (!U || !Bface) return fail(PLUTO_EINVAL, "null pointer");
    const Grid &g0 = C.dom[0].g;
    const int ndim = g0.ndim, nzl = C.nzloc;
    cudaStream_t s = C.stream;
    const size_t n = api_count(g0, nzl, -1);
    size_t nface = 0;
    for (int d = 0; d < ndim; d++) nface += api_count(g0, nzl, d);
    // Host arrays are staged on the device: U at offset 0, Bface behind it.  U[4..6], the cell-centred B of
    // the active dimensions, is never read (R7: it IS the face mean) and is not even copied; 2D: U[6] = B_z
    // goes to the third magnetic array.
    const double *dU = U, *dB = Bface;
    Staging st;
    if (!is_device_ptr(U) || !is_device_ptr(Bface)) {
        if (int rc = st.get(8 * n + nface)) return rc;
    }
    if (!is_device_ptr(U)) {
        CUDA_TRY(cudaMemcpyAsync(st.p, U, 4 * n * sizeof(double), cudaMemcpyHostToDevice, s));
        if (ndim == 2) CUDA_TRY(cudaMemcpyAsync(st.p + 6 * n, U + 6 * n, n * sizeof(double), cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaMemcpyAsync(st.p + 7 * n, U + 7 * n, n * sizeof(double), cudaMemcpyHostToDevice, s));
        dU = st.p;
    }
    if (!is_device_ptr(Bface)) {
        CUDA_TRY(cudaMemcpyAsync(st.p + 8 * n, Bface, nface * sizeof(double), cudaMemcpyHostToDevice, s));
        dB = st.p + 8 * n;
    }
    const int src_of[5] = { 0, 1, 2, 3, 7 };
    for (const Domain &d : C.dom) {
        const Grid &g = d.g;
        Box in = interior(g);
        for (int v = 0; v < 5; v++)
            k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dU + (size_t)src_of[v] * n, g.n[0], g.n[1], d.kz0, arr(d, A_SA + v));
        if (ndim == 2)
            k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dU + 6 * n, g.n[0], g.n[1], 0, arr(d, A_SA + S_B + 2));
        size_t off = 0;
        for (int f = 0; f < ndim; f++) {
            int m[3];
            api_extent(g0, nzl, f, m);
            k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dB + off, m[0], m[1], d.kz0, arr(d, A_SA + S_B + f));   // upper duplicates ignored
            off += api_count(g0, nzl, f);
        }
        C.launches += 5 + ndim + (ndim == 2 ? 1 : 0);
    }
    // every ghost once (the per-stage fill may skip x: see fill_ghosts); with peers the caller fills them
    // after all processes have set their state (pluto_fill_ghosts)
    if (peers_attached() && C.whole())
        for (const Domain &d : C.dom) fill_ghosts(d, A_SA, true);
    reset_bounds();
    StepParams p0;
    memset(&p0, 0, sizeof p0);
    CUDA_TRY(cudaMemcpyAsync(C.P, &p0, sizeof p0, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    C.have_state = true; C.stepped = false;
    return PLUTO_OK;
}

int pluto_fill_ghosts(void)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (!peers_attached()) return fail(PLUTO_ESTATE, "a neighbour slab is not attached (pluto_attach_peer)");
    for (const Domain &d : C.dom) fill_ghosts(d, A_SA, true);
    CUDA_TRY(cudaStreamSynchronize(C.stream));
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
}

int pluto_get_state(double *U, double *Bface)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (C.glm) return copy_state_glm(U, nullptr, false);
    if (!peers_attached()) return fail(PLUTO_ESTATE, "a neighbour slab is not attached (pluto_attach_peer)");
    const Grid &g0 = C.dom[0].g;
    const int ndim = g0.ndim, nzl = C.nzloc;
    cudaStream_t s = C.stream;
    const size_t n = api_count(g0, nzl, -1);
    size_t nface = 0;
    for (int d = 0; d < ndim; d++) nface += api_count(g0, nzl, d);
    Staging st;
    const bool udev = U && is_device_ptr(U), bdev = Bface && is_device_ptr(Bface);
    if ((U && !udev) || (Bface && !bdev)) {
        if (int rc = st.get(8 * n + nface)) return rc;
    }
    if (U) {
        double *dst = udev ? U : st.p;
        const int dst_of[5] = { 0, 1, 2, 3, 7 };
        for (const Domain &d : C.dom) {
            const Grid &g = d.g;
            Box in = interior(g);
            for (int v = 0; v < 5; v++)
                k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_SA + v), g.n[0], g.n[1], d.kz0, -1, dst + (size_t)dst_of[v] * n);
            k_pack_cellb<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_SA + S_B), peer_arr(d.nb[1], A_SA + S_B + 2), dst + 4 * n, (long long)n, d.kz0);
            C.launches += 6;
        }
        if (!udev) CUDA_TRY(cudaMemcpyAsync(U, dst, 8 * n * sizeof(double), cudaMemcpyDeviceToHost, s));
    }
    if (Bface) {
        double *dst = bdev ? Bface : st.p + 8 * n;      // behind U's staging: both copies overlap the packing
        for (const Domain &d : C.dom) {
            const Grid &g = d.g;
            size_t off = 0;
            for (int f = 0; f < ndim; f++) {
                int m[3];
                api_extent(g0, nzl, f, m);
                Box b = make_box(g, 0, g.n[0] + (f == 0), 0, g.n[1] + (f == 1), 0, g.n[2]);
                k_pack<<<grid_for(b), 128, 0, s>>>(g, b, arr(d, A_SA + S_B + f), m[0], m[1], d.kz0, -1, dst + off);
                if (f == 2 && &d == &C.dom.back()) {
                    // the duplicate upper z face of this process's planes: face 0 of the slab above
                    Box top = make_box(g, 0, g.n[0], 0, g.n[1], g.n[2], g.n[2] + 1);
                    k_pack<<<grid_for(top), 128, 0, s>>>(g, top, peer_arr(d.nb[1], A_SA + S_B + 2), m[0], m[1], d.kz0, 0, dst + off);
                    C.launches += 1;
                }
                off += api_count(g0, nzl, f);
            }
            C.launches += ndim;
        }
        if (!bdev) CUDA_TRY(cudaMemcpyAsync(Bface, dst, nface * sizeof(double), cudaMemcpyDeviceToHost, s));
    }
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
}

int pluto_set_psi(const double *psi)
{
    if (!C.init || !C.have_state || !C.glm) return fail(PLUTO_ESTATE, "needs a state of the GLM variant");
    if (!psi) return fail(PLUTO_EINVAL, "null pointer");
    return copy_state_glm(nullptr, const_cast<double *>(psi), true);
}

int pluto_get_psi(double *psi)
{
    if (!C.init || !C.have_state || !C.glm) return fail(PLUTO_ESTATE, "needs a state of the GLM variant");
    if (!psi) return fail(PLUTO_EINVAL, "null pointer");
    return copy_state_glm(nullptr, psi, false);
}

int pluto_step_async(int nsteps)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (nsteps < 0) return fail(PLUTO_EINVAL, "nsteps < 0");
    return run_steps(nsteps, false);
}

int pluto_sync(void)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    return finish();
}

int pluto_step(int nsteps)
{
    int rc = pluto_step_async(nsteps);
    return rc ? rc : finish();
}

int pluto_step_fixed_dt(int nsteps, double dt)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (nsteps < 0 || !(dt > 0.0)) return fail(PLUTO_EINVAL, "need nsteps >= 0 and dt > 0");
    CUDA_TRY(cudaMemcpyAsync(&C.P->dt_fixed, &dt, sizeof dt, cudaMemcpyHostToDevice, C.stream));
    CUDA_TRY(cudaStreamSynchronize(C.stream));
    int rc = run_steps(nsteps, true);
    return rc ? rc : finish();
}

// ---- the step in phases, for a box whose slabs live in several processes (one per GPU)

int pluto_step_begin(double fixed_dt)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (!peers_attached()) return fail(PLUTO_ESTATE, "a neighbour slab is not attached (pluto_attach_peer)");
    if (int rc = ensure_rk3_storage()) return rc;
    if (int rc = ensure_uct_storage()) return rc;
    if (fixed_dt > 0.0) {
        CUDA_TRY(cudaMemcpyAsync(&C.P->dt_fixed, &fixed_dt, sizeof fixed_dt, cudaMemcpyHostToDevice, C.stream));
        CUDA_TRY(cudaStreamSynchronize(C.stream));
    } else {
        enqueue_dtmax(false);
    }
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
}

void *pluto_dt_max_bits(void) { return C.init ? (void *)&C.P->smax_bits : nullptr; }

int pluto_step_stage(int stage, int fixed)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (stage < 0 || stage >= C.rk_order) return fail(PLUTO_EINVAL, "stage out of range");
    // a stage without its pluto_step_begin, or an option switched in between: the stage kernels would read a
    // neighbour that is not there, or work arrays that were never allocated
    if (!peers_attached()) return fail(PLUTO_ESTATE, "a neighbour slab is not attached (pluto_attach_peer)");
    if (int rc = ensure_rk3_storage()) return rc;
    if (int rc = ensure_uct_storage()) return rc;
    if (stage == 0) LAUNCH(K_SCALAR, launch_dtfinish(C.dom[0].g, C.P, fixed ? 1 : 0, C.stream));
    enqueue_rk_stage(stage);
    if (stage == C.rk_order - 1) {
        LAUNCH(K_SCALAR, launch_advance_time(C.P, C.stream));
        C.stepped = true;
    }
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
}

double pluto_get_dt(void)
{
    if (!C.init || !C.have_state) return NAN;
    double dt = NAN;
    if (!C.stepped) {
        if (!C.whole()) return NAN;             // the max over every process is the caller's (pluto_dt_max_bits)
        enqueue_dt(2);
        if (cudaMemcpyAsync(&dt, &C.P->dt_probe, sizeof dt, cudaMemcpyDeviceToHost, C.stream) != cudaSuccess) return NAN;
    } else {
        if (cudaMemcpyAsync(&dt, &C.P->dt, sizeof dt, cudaMemcpyDeviceToHost, C.stream) != cudaSuccess) return NAN;
    }
    if (cudaStreamSynchronize(C.stream) != cudaSuccess) return NAN;
    return dt;
}

double pluto_get_time(void)
{
    if (!C.init || !C.have_state) return NAN;
    double t = NAN;
    if (cudaMemcpyAsync(&t, &C.P->time, sizeof t, cudaMemcpyDeviceToHost, C.stream) != cudaSuccess) return NAN;
    if (cudaStreamSynchronize(C.stream) != cudaSuccess) return NAN;
    return t;
}

long long pluto_launch_count(void) { return C.launches; }
long long pluto_graph_captures(void) { return C.captures; }

int pluto_profile(int on)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (on) {
        const size_t pairs = 8192;
        while (C.prof_ev.size() < 2 * pairs) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreate(&e));
            C.prof_ev.push_back(e);
        }
        C.prof_kid.assign(pairs, 0);
        CUDA_TRY(cudaStreamSynchronize(C.stream));
        C.prof_used = 0;
        for (int k = 0; k < K_COUNT; k++) { C.prof_ms[k] = 0.0; C.prof_cnt[k] = 0; }
        C.prof_on = true;
    } else if (C.prof_on) {
        prof_flush();
        C.prof_on = false;
    }
    return PLUTO_OK;
}

int pluto_profile_get(int kernel, double *total_ms, long long *launches)
{
    if (kernel < 0 || kernel >= K_COUNT) return fail(PLUTO_EINVAL, "kernel id out of range");
    if (C.prof_on) prof_flush();
    if (total_ms) *total_ms = C.prof_ms[kernel];
    if (launches) *launches = C.prof_cnt[kernel];
    return PLUTO_OK;
}

const char *pluto_kernel_name(int kernel)
{
    return (kernel < 0 || kernel >= K_COUNT) ? nullptr : kKernelNames[kernel];
}

double pluto_probe_fp64_gflops(void)
{
    if (pluto_device_count() < 1) { fail(PLUTO_ECUDA, "no CUDA device"); return NAN; }
    return pluto::probe_fp64_gflops(C.stream);
}

int pluto_debug_euler(double dt, double *U1, double *Bf1, double *W, double *Fem, double *Eedge)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    if (C.dom.size() != 1 || !C.whole() || C.glm) return fail(PLUTO_ESTATE, "pluto_debug_euler works on a single domain of the CT scheme");
    if (!(dt > 0.0)) return fail(PLUTO_EINVAL, "dt must be positive");
    // in UCT-HLLD mode the CT work arrays hold the a / d coefficients and transverse velocities of R19 instead of
    // the upwind weight and the two induction fluxes: there is no W or Fem to hand out
    if (C.emf == 1 && (W || Fem)) return fail(PLUTO_ESTATE, "pluto_debug_euler: W and Fem do not exist in UCT-HLLD mode (pass NULL)");
    if (int rc = ensure_uct_storage()) return rc;
    const Domain &d = C.dom[0];
    const Grid &g = d.g;
    cudaStream_t s = C.stream;
    CUDA_TRY(cudaMemcpyAsync(&C.P->dt_fixed, &dt, sizeof dt, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    // keep dt/time of the real run intact: save and restore the scalars
    StepParams saved;
    CUDA_TRY(cudaMemcpy(&saved, C.P, sizeof saved, cudaMemcpyDeviceToHost));
    launch_dtfinish(g, C.P, 1, s);
    // two library-owned temporaries, freed on every path: the edge EMFs (never stored by the production
    // path) and a private staging area (the CT work arrays are being read)
    struct DevBuf {
        double *p = nullptr;
        ~DevBuf() { if (p) cudaFree(p); }
    } dbgE, tmpb;
    CUDA_TRY(cudaMalloc((void **)&dbgE.p, 3 * (size_t)g.sa * sizeof(double)));
    CUDA_TRY(cudaMemsetAsync(dbgE.p, 0, 3 * (size_t)g.sa * sizeof(double), s));
    enqueue_stage(A_SA, A_SB, -1, 0.0, 1.0, false, dbgE.p);
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    const size_t n = api_count(g, g.n[2], -1);
    size_t maxcount = 8 * n + 3 * (n + (size_t)g.n[0] * g.n[1] + (size_t)g.n[1] * g.n[2] + (size_t)g.n[0] * g.n[2]);
    CUDA_TRY(cudaMalloc((void **)&tmpb.p, maxcount * sizeof(double)));
    double *tmp = tmpb.p;
    Box in = interior(g);
    auto emit = [&](double *user, size_t count) -> int {
        if (is_device_ptr(user)) return cudaMemcpy(user, tmp, count * sizeof(double), cudaMemcpyDeviceToDevice) == cudaSuccess ? 0 : 1;
        return cudaMemcpy(user, tmp, count * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : 1;
    };
    int bad = 0;
    if (U1) {
        const int dst_of[5] = { 0, 1, 2, 3, 7 };
        for (int v = 0; v < 5; v++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_SB + v), g.n[0], g.n[1], 0, -1, tmp + dst_of[v] * n);
        k_pack_cellb<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_SB + S_B), arr(d, A_SB + S_B + 2), tmp + 4 * n, (long long)n, 0);
        cudaStreamSynchronize(s);
        bad |= emit(U1, 8 * n);
    }
    if (Bf1) {
        size_t off = 0;
        for (int f = 0; f < g.ndim; f++) {
            int m[3];
            api_extent(g, g.n[2], f, m);
            Box b = make_box(g, 0, m[0], 0, m[1], 0, g.n[2]);
            k_pack<<<grid_for(b), 128, 0, s>>>(g, b, arr(d, A_SB + S_B + f), m[0], m[1], 0, -1, tmp + off);
            if (f == 2) {
                Box top = make_box(g, 0, g.n[0], 0, g.n[1], g.n[2], g.n[2] + 1);
                k_pack<<<grid_for(top), 128, 0, s>>>(g, top, arr(d, A_SB + S_B + 2), m[0], m[1], 0, 0, tmp + off);
            }
            off += api_count(g, g.n[2], f);
        }
        cudaStreamSynchronize(s);
        bad |= emit(Bf1, off);
    }
    if (W) {
        cudaMemsetAsync(tmp, 0, 3 * n * sizeof(double), s);
        for (int f = 0; f < g.ndim; f++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_CT + CT_W + f), g.n[0], g.n[1], 0, -1, tmp + f * n);
        cudaStreamSynchronize(s);
        bad |= emit(W, 3 * n);
    }
    if (Fem) {
        cudaMemsetAsync(tmp, 0, 6 * n * sizeof(double), s);
        for (int f = 0; f < g.ndim; f++)
            for (int q = 0; q < 2; q++)
                k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(d, A_CT + CT_FEM + 2 * f + q), g.n[0], g.n[1], 0, -1, tmp + (2 * f + q) * n);
        cudaStreamSynchronize(s);
        bad |= emit(Fem, 6 * n);
    }
    if (Eedge) {
        cudaMemsetAsync(tmp, 0, 3 * n * sizeof(double), s);
        for (int e = (g.act[2] ? 0 : 2); e < 3; e++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, dbgE.p + (size_t)e * g.sa, g.n[0], g.n[1], 0, -1, tmp + e * n);
        cudaStreamSynchronize(s);
        bad |= emit(Eedge, 3 * n);
    }
    int err = 0;
    CUDA_TRY(cudaMemcpy(&err, &C.P->err, sizeof(int), cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(C.P, &saved, sizeof saved, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaGetLastError());
    if (bad) return fail(PLUTO_ECUDA, "debug copy failed");
    return err ? PLUTO_EPHYS : PLUTO_OK;
}

} // extern "C"
