// pluto_api.cu -- the C-ABI of include/pluto.h: context, memory, host<->device copies, and the
// launch sequence of one RK2 step.  No CPU fallback: without a device every call fails loudly.
#include "../../include/pluto.h"
#include "kernels.cuh"
#include "ct_tma.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

namespace pluto {
void launch_dtmax(const Grid &g, const double *U, StepParams *P, int nblocks, cudaStream_t s);
void launch_dtfinish(const Grid &g, StepParams *P, int mode, cudaStream_t s);
void launch_advance_time(StepParams *P, cudaStream_t s);
double probe_fp64_gflops(cudaStream_t s);
}

using namespace pluto;

namespace {

enum KernelId { K_GHOST = 0, K_FLUX_XY, K_FLUX_X, K_FLUX_Y, K_FLUX_Z, K_CT, K_DTMAX, K_SCALAR, K_PACK, K_CT_HALO, K_COUNT };
const char *const kKernelNames[K_COUNT] = { "ghost_fill", "sweep_xy", "sweep_x", "sweep_y", "sweep_z", "ct",
                                            "dt_max", "scalars", "pack_unpack", "ct_halo" };

struct Context {
    bool init = false;
    bool have_state = false;
    bool stepped = false;
    Grid g{};
    double *base = nullptr;          // A_COUNT arrays
    StepParams *P = nullptr;         // device scalars (inside the allocation)
    bool own_mem = false;
    void *ws = nullptr;              // registered workspace
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;   // stream in use (the caller's, or own_stream)
    cudaStream_t own_stream = nullptr;
    long long launches = 0;
    long long per_step[2] = { 0, 0 };
    int use_graph = 1;
    int fuse_xy = 1;
    int ct_tma = 1;
    int rk_order = 2;                // 2: SSP-RK2 (R3), 3: SSP-RK3 (Eq. 5)
    CUtensorMap ct_map{};            // the twelve CT arrays as one 4D tensor (x, y, z, array)
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

double *arr(int id) { return C.base + (long long)id * C.g.sa; }

size_t layout_bytes(const Grid &g) { return (size_t)A_COUNT * g.sa * sizeof(double) + 256; }

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

// TMA descriptor of the CT work arrays: dims (pitch, tot1, tot2, CT_COUNT) doubles, box = one tile of
// one array.  cuTensorMapEncodeTiled is taken from the driver through the runtime (no -lcuda).
int make_ct_map()
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
    const Grid &g = C.g;
    cuuint64_t dims[4] = { (cuuint64_t)g.tot[0], (cuuint64_t)g.tot[1], (cuuint64_t)g.tot[2], (cuuint64_t)CT_COUNT };
    cuuint64_t strides[3] = { (cuuint64_t)g.st[1] * 8, (cuuint64_t)g.st[2] * 8, (cuuint64_t)g.sa * 8 };
    cuuint32_t box[4] = { CTM_COLS, CTM_ROWS, 1, 1 }, estr[4] = { 1, 1, 1, 1 };
    CUresult r = encode(&C.ct_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, arr(A_CT), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(PLUTO_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
    return PLUTO_OK;
}

// ---------------------------------------------------------------- launch sequences

// ghost layers of the 8 arrays of one state, one launch
// widths for which the fused x+y sweep spans a whole periodic row: no kernel then reads an x ghost
// other than the x-face n0 (kept equal to face 0 by the CT kernel)
bool row_wraps(int nx) { return nx == 64 || nx == 128 || nx == 256 || nx == 512; }

void fill_ghosts(double *state, bool all = false)
{
    const Grid &g = C.g;
    if (!all && C.fuse_xy && g.limiter != 2 && row_wraps(g.n[0])) {
        const int ngh = 2 * g.ng + 1;
        const int rows = (g.act[2] ? ngh * (g.n[1] + ngh) : 0) + g.n[2] * ngh;
        LAUNCH(K_GHOST, k_ghost_yz<<<dim3(rows, S_COUNT), 128, 0, C.stream>>>(g, state));
    } else {
        LAUNCH(K_GHOST, k_ghost<<<C.sm_count * 8, 256, 0, C.stream>>>(g, state, S_COUNT));
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

template <int LIM, bool TWO_D>
void launch_sweeps(const double *Sin, double *Sout, Combine cb)
{
    const Grid &g = C.g;
    cudaStream_t s = C.stream;
    double *ct = arr(A_CT);
    const double scale = cb.Sn ? cb.ws : 1.0;
    bool fused = false;
    if constexpr (LIM != 2) if (C.fuse_xy) {
        fused = true;
        // fused x + y sweep: one block per x-row chunk and y-segment.  The block width is a template
        // parameter (shared-memory offsets become immediates): a whole periodic row when nx is one of
        // the instantiated widths, else chunks of 128 or 256 threads that overlap by four cells.
        const int nx = g.n[0];
        const bool wrap = row_wraps(nx);
        const int nt = wrap ? nx : (nx > 124 ? 256 : 128);
        const int chunks = wrap ? 1 : (nx + nt - 5) / (nt - 4);
        const int len = march_seglen(g.n[1], (long long)nx * g.n[2]);
        dim3 grid(chunks, (g.n[1] + len - 1) / len, g.n[2]);
        const size_t smem = (size_t)XY_DOUBLES_PER_THREAD * nt * sizeof(double) + XY_SMEM_EXTRA(nt);
        void (*k)(Grid, const double *, double *, double *, StepParams *, Combine, int) =
            wrap ? (nt == 64 ? k_sweep_xy<LIM, TWO_D, true, 64> : nt == 128 ? k_sweep_xy<LIM, TWO_D, true, 128>
                    : nt == 256 ? k_sweep_xy<LIM, TWO_D, true, 256> : k_sweep_xy<LIM, TWO_D, true, 512>)
                 : (nt == 128 ? k_sweep_xy<LIM, TWO_D, false, 128> : k_sweep_xy<LIM, TWO_D, false, 256>);
        cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        LAUNCH(K_FLUX_XY, k<<<grid, nt, smem, s>>>(g, Sin, Sout, ct, C.P, cb, len));
    }
    if (!fused) {
        if constexpr (LIM == 2) {
            cudaFuncSetAttribute(k_sweep_march_wz<1, TWO_D>, cudaFuncAttributeMaxDynamicSharedMemorySize, WZ_SMEM_BYTES);
            cudaFuncSetAttribute(k_sweep_march_wz<2, TWO_D>, cudaFuncAttributeMaxDynamicSharedMemorySize, WZ_SMEM_BYTES);
        }
        const long long nitems = (long long)(g.n[0] + 2 * sx_halo(LIM)) * g.n[1] * g.n[2];
        LAUNCH(K_FLUX_X, k_sweep_x<LIM, TWO_D><<<(unsigned)((nitems + sx_out(LIM) - 1) / sx_out(LIM)), SX_NT, 0, s>>>(
                             g, Sin, Sout, ct, C.P, cb));
        const int bx = (g.n[0] + MARCH_NT - 1) / MARCH_NT;
        const int len = march_seglen(g.n[1], (long long)g.n[0] * g.n[2]);
        dim3 grid(bx, (g.n[1] + len - 1) / len, g.n[2]);
        if constexpr (LIM == 2) LAUNCH(K_FLUX_Y, k_sweep_march_wz<1, TWO_D><<<grid, MARCH_NT, WZ_SMEM_BYTES, s>>>(g, Sin, Sout, ct, C.P, scale, len));
        else LAUNCH(K_FLUX_Y, k_sweep_march<1, LIM, TWO_D><<<grid, MARCH_NT, 0, s>>>(g, Sin, Sout, ct, C.P, scale, len));
    }
    if (!TWO_D) {
        const int bx = (g.n[0] + MARCH_NT - 1) / MARCH_NT;
        const int len = march_seglen(g.n[2], (long long)g.n[0] * g.n[1]);
        dim3 grid(bx, g.n[1], (g.n[2] + len - 1) / len);
        if constexpr (LIM == 2) LAUNCH(K_FLUX_Z, k_sweep_march_wz<2, TWO_D><<<grid, MARCH_NT, WZ_SMEM_BYTES, s>>>(g, Sin, Sout, ct, C.P, scale, len));
        else LAUNCH(K_FLUX_Z, k_sweep_march<2, LIM, TWO_D><<<grid, MARCH_NT, 0, s>>>(g, Sin, Sout, ct, C.P, scale, len));
    }
}

// CT: edge EMFs + face update (+ combine) in one kernel; dbg (debug only) receives the edge EMFs
void launch_ct(const double *bin, double *bout, Combine cb, double *dbg)
{
    const bool combine = cb.Sn != nullptr;
    const Grid &g = C.g;
    cudaStream_t s = C.stream;
    const int tiles_x = (g.n[0] + CT_TX - 2) / (CT_TX - 1), tiles_y = (g.n[1] + CT_TY - 2) / (CT_TY - 1);
    const int len = march_seglen(g.n[2], (long long)tiles_x * tiles_y * CT_TX * CT_TY);
    dim3 grid(tiles_x, tiles_y, (g.n[2] + len - 1) / len), block(CT_TX, CT_TY);
    const double *ct = arr(A_CT);
    if (C.ct_tma) {
        // periodic halo layer of the CT arrays, then the TMA-staged kernel
        LAUNCH(K_CT_HALO, k_ct_halo<<<dim3(g.n[2], CT_COUNT), 256, 0, s>>>(g, arr(A_CT), g.act[2] ? 0 : 1));
        static bool tma_attr = false;
        if (!tma_attr) {
            cudaFuncSetAttribute(k_ct_tma<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES);
            cudaFuncSetAttribute(k_ct_tma<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES);
            cudaFuncSetAttribute(k_ct_tma<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES);
            cudaFuncSetAttribute(k_ct_tma<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, CTM_SMEM_BYTES);
            tma_attr = true;
        }
        if (g.act[2]) {
            if (combine) LAUNCH(K_CT, k_ct_tma<true, false><<<grid, block, CTM_SMEM_BYTES, s>>>(g, C.ct_map, ct, bin, bout, C.P, len, dbg, cb));
            else         LAUNCH(K_CT, k_ct_tma<false, false><<<grid, block, CTM_SMEM_BYTES, s>>>(g, C.ct_map, ct, bin, bout, C.P, len, dbg, cb));
        } else {
            if (combine) LAUNCH(K_CT, k_ct_tma<true, true><<<grid, block, CTM_SMEM_BYTES, s>>>(g, C.ct_map, ct, bin, bout, C.P, len, dbg, cb));
            else         LAUNCH(K_CT, k_ct_tma<false, true><<<grid, block, CTM_SMEM_BYTES, s>>>(g, C.ct_map, ct, bin, bout, C.P, len, dbg, cb));
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

// One Runge-Kutta stage: Sout <- Euler(Sin), or with a combine  Sout <- wn * S^n + ws * Euler(Sin)
// (sn < 0: no combine; sn may equal out: in place).
void enqueue_stage(int in, int out, int sn = -1, double wn = 0.0, double ws = 1.0, double *dbg = nullptr)
{
    const Grid &g = C.g;
    fill_ghosts(arr(in));
    const bool two_d = !g.act[2];
    const Combine cb = { sn >= 0 ? arr(sn) : nullptr, wn, ws };
    if (g.limiter == 0)      { if (two_d) launch_sweeps<0, true>(arr(in), arr(out), cb);
                               else       launch_sweeps<0, false>(arr(in), arr(out), cb); }
    else if (g.limiter == 1) { if (two_d) launch_sweeps<1, true>(arr(in), arr(out), cb);
                               else       launch_sweeps<1, false>(arr(in), arr(out), cb); }
    else                     { if (two_d) launch_sweeps<2, true>(arr(in), arr(out), cb);
                               else       launch_sweeps<2, false>(arr(in), arr(out), cb); }
    const Combine cbf = { sn >= 0 ? arr(sn + S_B) : nullptr, wn, ws };
    launch_ct(arr(in + S_B), arr(out + S_B), cbf, dbg);
}

void enqueue_dt(int mode)
{
    if (mode != 1) LAUNCH(K_DTMAX, launch_dtmax(C.g, arr(A_SA), C.P, C.sm_count * 8, C.stream));
    LAUNCH(K_SCALAR, launch_dtfinish(C.g, C.P, mode, C.stream));
}

void enqueue_step(bool fixed)
{
    enqueue_dt(fixed ? 1 : 0);
    if (C.rk_order == 3) {
        // SSP-RK3, Eq. 5 (R17: the last stage carries 2 L**)
        enqueue_stage(A_SA, A_SB);                                  // S*   = S^n + L(S^n)
        enqueue_stage(A_SB, A_SC, A_SA, 0.75, 0.25);                // S**  = (3 S^n + S* + L(S*)) / 4
        enqueue_stage(A_SC, A_SA, A_SA, 1.0 / 3.0, 2.0 / 3.0);      // S^{n+1} = (S^n + 2 (S** + L(S**))) / 3
    } else {
        enqueue_stage(A_SA, A_SB);                                  // S^1 = S^n + L(S^n)
        enqueue_stage(A_SB, A_SA, A_SA, 0.5, 0.5);                  // S^{n+1} = (S^n + S^1 + L(S^1)) / 2
    }
    LAUNCH(K_SCALAR, launch_advance_time(C.P, C.stream));
}

int run_steps(int nsteps, bool fixed)
{
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

// extents of the caller's array for the face family d (d = -1: cell array)
void api_extent(const Grid &g, int d, int m[3])
{
    for (int a = 0; a < 3; a++) m[a] = g.n[a] + (a == d ? 1 : 0);
}

size_t api_count(const Grid &g, int d)
{
    int m[3];
    api_extent(g, d, m);
    return (size_t)m[0] * m[1] * m[2];
}

// staging buffer: the CT work arrays are free outside a step (12 padded arrays > 11 interior arrays)
double *staging() { return arr(A_CT); }

} // namespace

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
    Grid g;
    if (!make_grid(g, nx, ny, nz, ghost)) return 0;
    return layout_bytes(g);
}

int pluto_set_workspace(void *dev, size_t bytes)
{
    if (C.init && !C.own_mem) return fail(PLUTO_ESTATE, "workspace in use: call pluto_finalize first");
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
        // the legacy default stream cannot be captured into a graph: use a stream of our own
        if (!C.own_stream && pluto_device_count() > 0)
            if (cudaStreamCreateWithFlags(&C.own_stream, cudaStreamNonBlocking) != cudaSuccess) {
                cudaGetLastError();
                return fail(PLUTO_ECUDA, "cannot create a stream");
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
    if (C.init) {
        cudaStreamSynchronize(C.stream);
        destroy_graphs();
        if (C.own_mem && C.base) cudaFree(C.base);
    }
    C.base = nullptr; C.P = nullptr; C.init = false; C.have_state = false; C.stepped = false; C.own_mem = false;
    return PLUTO_OK;
}

int pluto_init(int nx, int ny, int nz, int ghost, double gamma, double cfl, int limiter)
{
    if (pluto_device_count() < 1) return fail(PLUTO_ECUDA, "no CUDA device: this library has no CPU fallback");
    pluto_finalize();
    if (!C.stream) { int rc = pluto_set_stream(nullptr); if (rc) return rc; }
    Grid g;
    if (!make_grid(g, nx, ny, nz, ghost))
        return fail(PLUTO_EINVAL, "need nx >= 2, ny >= 2, nz >= 1, 2 <= ghost <= %d, active extents >= ghost", XOFF);
    if (!(gamma > 1.0) || !(cfl > 0.0) || limiter < PLUTO_MINMOD || limiter > PLUTO_WENOZ)
        return fail(PLUTO_EINVAL, "need gamma > 1, cfl > 0, limiter in {0,1,2}");
    if (limiter == PLUTO_WENOZ && ghost < 3)
        return fail(PLUTO_EINVAL, "the WENO-Z stencil needs ghost >= 3");
    if ((long long)g.tot[2] * 8 > 65535 || g.tot[1] > 65535)
        return fail(PLUTO_EINVAL, "extent too large for the launch grid");
    g.gamma = gamma; g.igm1 = 1.0 / (gamma - 1.0); g.cfl = cfl; g.limiter = limiter;
    for (int a = 0; a < 3; a++) { g.dx[a] = 1.0 / nx; g.idx[a] = 1.0 / g.dx[a]; }   // R11: Lx = 1, cubic cells
    size_t bytes = layout_bytes(g);
    if (C.ws) {
        if (C.ws_bytes < bytes) return fail(PLUTO_ENOMEM, "workspace has %zu bytes, need %zu", C.ws_bytes, bytes);
        C.base = (double *)C.ws;
        C.own_mem = false;
    } else {
        cudaError_t e = cudaMalloc((void **)&C.base, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); C.base = nullptr; return fail(PLUTO_ENOMEM, "cudaMalloc(%zu): %s", bytes, cudaGetErrorString(e)); }
        C.own_mem = true;
    }
    C.g = g;
    C.P = (StepParams *)(C.base + (long long)A_COUNT * g.sa);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&C.sm_count, cudaDevAttrMultiProcessorCount, dev);
    CUDA_TRY(cudaMemsetAsync(C.base, 0, bytes, C.stream));
    CUDA_TRY(cudaStreamSynchronize(C.stream));
    C.init = true; C.have_state = false; C.stepped = false; C.launches = 0;
    int rc = make_ct_map();
    if (rc) { C.init = false; return rc; }
    return PLUTO_OK;
}

int pluto_set_box(double Lx, double Ly, double Lz)
{
    if (!C.init) return fail(PLUTO_ESTATE, "not initialised");
    if (!(Lx > 0.0) || !(Ly > 0.0) || !(Lz > 0.0)) return fail(PLUTO_EINVAL, "box lengths must be positive");
    double L[3] = { Lx, Ly, Lz };
    for (int a = 0; a < 3; a++) { C.g.dx[a] = L[a] / C.g.n[a]; C.g.idx[a] = 1.0 / C.g.dx[a]; }
    destroy_graphs();          // kernels take the grid by value: captured copies are stale
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
    if (!U || !Bface) return fail(PLUTO_EINVAL, "null pointer");
    const Grid &g = C.g;
    cudaStream_t s = C.stream;
    Box in = interior(g);
    const size_t n = api_count(g, -1);
    size_t nface = 0;
    for (int d = 0; d < g.ndim; d++) nface += api_count(g, d);
    // Host arrays are staged in the CT work arrays (free outside a step): U at offset 0, Bface behind it.
    // U[4..6], the cell-centred B of the active dimensions, is never read (R7: it IS the face mean) and
    // is not even copied; 2D: U[6] = B_z goes to the third magnetic array.
    const double *dU = U, *dB = Bface;
    if (!is_device_ptr(U)) {
        if ((8 * n + nface) * sizeof(double) > (size_t)CT_COUNT * g.sa * sizeof(double)) return fail(PLUTO_ENOMEM, "staging too small");
        CUDA_TRY(cudaMemcpyAsync(staging(), U, 4 * n * sizeof(double), cudaMemcpyHostToDevice, s));
        if (!g.act[2]) CUDA_TRY(cudaMemcpyAsync(staging() + 6 * n, U + 6 * n, n * sizeof(double), cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaMemcpyAsync(staging() + 7 * n, U + 7 * n, n * sizeof(double), cudaMemcpyHostToDevice, s));
        dU = staging();
    }
    if (!is_device_ptr(Bface)) {
        if ((8 * n + nface) * sizeof(double) > (size_t)CT_COUNT * g.sa * sizeof(double)) return fail(PLUTO_ENOMEM, "staging too small");
        CUDA_TRY(cudaMemcpyAsync(staging() + 8 * n, Bface, nface * sizeof(double), cudaMemcpyHostToDevice, s));
        dB = staging() + 8 * n;
    }
    const int src_of[5] = { 0, 1, 2, 3, 7 };
    for (int v = 0; v < 5; v++)
        k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dU + (size_t)src_of[v] * n, g.n[0], g.n[1], arr(A_SA + v));
    if (!g.act[2])
        k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dU + 6 * n, g.n[0], g.n[1], arr(A_SA + S_B + 2));
    const double *dev = dB;
    size_t off = 0;
    for (int d = 0; d < g.ndim; d++) {
        int m[3];
        api_extent(g, d, m);
        k_unpack<<<grid_for(in), 128, 0, s>>>(g, in, dev + off, m[0], m[1], arr(A_SA + S_B + d));   // upper duplicate ignored
        off += api_count(g, d);
    }
    fill_ghosts(arr(A_SA), true);    // every ghost once (the per-stage fill may skip x: see fill_ghosts)
    StepParams p0;
    memset(&p0, 0, sizeof p0);
    CUDA_TRY(cudaMemcpyAsync(C.P, &p0, sizeof p0, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    C.launches += 6 + g.ndim;
    C.have_state = true; C.stepped = false;
    return PLUTO_OK;
}

int pluto_get_state(double *U, double *Bface)
{
    if (!C.init || !C.have_state) return fail(PLUTO_ESTATE, "no state");
    const Grid &g = C.g;
    cudaStream_t s = C.stream;
    const size_t n = api_count(g, -1);
    if (U) {
        bool dev = is_device_ptr(U);
        double *dst = dev ? U : staging();
        Box in = interior(g);
        const int dst_of[5] = { 0, 1, 2, 3, 7 };
        for (int v = 0; v < 5; v++)
            k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_SA + v), g.n[0], g.n[1], dst + (size_t)dst_of[v] * n);
        k_pack_cellb<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_SA + S_B), dst + 4 * n, (long long)n);
        if (!dev) CUDA_TRY(cudaMemcpyAsync(U, dst, 8 * n * sizeof(double), cudaMemcpyDeviceToHost, s));
        C.launches += 6;
    }
    if (Bface) {
        bool dev = is_device_ptr(Bface);
        double *dst = dev ? Bface : staging() + 8 * n;      // behind U's staging: both copies overlap the packing
        size_t off = 0;
        for (int d = 0; d < g.ndim; d++) {
            int m[3];
            api_extent(g, d, m);
            Box b = make_box(g, 0, m[0], 0, m[1], 0, m[2]);
            k_pack<<<grid_for(b), 128, 0, s>>>(g, b, arr(A_SA + S_B + d), m[0], m[1], dst + off);
            off += api_count(g, d);
        }
        if (!dev) CUDA_TRY(cudaMemcpyAsync(Bface, dst, off * sizeof(double), cudaMemcpyDeviceToHost, s));
        C.launches += g.ndim;
    }
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    return PLUTO_OK;
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

double pluto_get_dt(void)
{
    if (!C.init || !C.have_state) return NAN;
    double dt = NAN;
    if (!C.stepped) {
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
    if (!(dt > 0.0)) return fail(PLUTO_EINVAL, "dt must be positive");
    const Grid &g = C.g;
    cudaStream_t s = C.stream;
    CUDA_TRY(cudaMemcpyAsync(&C.P->dt_fixed, &dt, sizeof dt, cudaMemcpyHostToDevice, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    // keep dt/time of the real run intact: save and restore the scalars
    StepParams saved;
    CUDA_TRY(cudaMemcpy(&saved, C.P, sizeof saved, cudaMemcpyDeviceToHost));
    launch_dtfinish(g, C.P, 1, s);
    double *dbgE = nullptr;                     // edge EMFs are never stored by the production path
    CUDA_TRY(cudaMalloc((void **)&dbgE, 3 * (size_t)g.sa * sizeof(double)));
    CUDA_TRY(cudaMemsetAsync(dbgE, 0, 3 * (size_t)g.sa * sizeof(double), s));
    enqueue_stage(A_SA, A_SB, -1, 0.0, 1.0, dbgE);
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    const size_t n = api_count(g, -1);
    double *tmp = nullptr;                      // private staging: the flux arrays are being read
    size_t maxcount = 8 * n + 3 * (n + (size_t)g.n[0] * g.n[1] + (size_t)g.n[1] * g.n[2] + (size_t)g.n[0] * g.n[2]);
    CUDA_TRY(cudaMalloc((void **)&tmp, maxcount * sizeof(double)));
    Box in = interior(g);
    auto emit = [&](double *user, size_t count) -> int {
        if (is_device_ptr(user)) return cudaMemcpy(user, tmp, count * sizeof(double), cudaMemcpyDeviceToDevice) == cudaSuccess ? 0 : 1;
        return cudaMemcpy(user, tmp, count * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess ? 0 : 1;
    };
    int bad = 0;
    if (U1) {
        const int dst_of[5] = { 0, 1, 2, 3, 7 };
        for (int v = 0; v < 5; v++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_SB + v), g.n[0], g.n[1], tmp + dst_of[v] * n);
        k_pack_cellb<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_SB + S_B), tmp + 4 * n, (long long)n);
        cudaStreamSynchronize(s);
        bad |= emit(U1, 8 * n);
    }
    if (Bf1) {
        size_t off = 0;
        for (int d = 0; d < g.ndim; d++) {
            int m[3];
            api_extent(g, d, m);
            Box b = make_box(g, 0, m[0], 0, m[1], 0, m[2]);
            k_pack<<<grid_for(b), 128, 0, s>>>(g, b, arr(A_SB + S_B + d), m[0], m[1], tmp + off);
            off += api_count(g, d);
        }
        cudaStreamSynchronize(s);
        bad |= emit(Bf1, off);
    }
    if (W) {
        cudaMemsetAsync(tmp, 0, 3 * n * sizeof(double), s);
        for (int d = 0; d < g.ndim; d++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_CT + CT_W + d), g.n[0], g.n[1], tmp + d * n);
        cudaStreamSynchronize(s);
        bad |= emit(W, 3 * n);
    }
    if (Fem) {
        cudaMemsetAsync(tmp, 0, 6 * n * sizeof(double), s);
        for (int d = 0; d < g.ndim; d++)
            for (int q = 0; q < 2; q++)
                k_pack<<<grid_for(in), 128, 0, s>>>(g, in, arr(A_CT + CT_FEM + 2 * d + q), g.n[0], g.n[1], tmp + (2 * d + q) * n);
        cudaStreamSynchronize(s);
        bad |= emit(Fem, 6 * n);
    }
    if (Eedge) {
        cudaMemsetAsync(tmp, 0, 3 * n * sizeof(double), s);
        for (int e = (g.act[2] ? 0 : 2); e < 3; e++) k_pack<<<grid_for(in), 128, 0, s>>>(g, in, dbgE + (size_t)e * g.sa, g.n[0], g.n[1], tmp + e * n);
        cudaStreamSynchronize(s);
        bad |= emit(Eedge, 3 * n);
    }
    cudaFree(dbgE);
    cudaFree(tmp);
    int err = 0;
    CUDA_TRY(cudaMemcpy(&err, &C.P->err, sizeof(int), cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(C.P, &saved, sizeof saved, cudaMemcpyHostToDevice));
    CUDA_TRY(cudaGetLastError());
    if (bad) return fail(PLUTO_ECUDA, "debug copy failed");
    return err ? PLUTO_EPHYS : PLUTO_OK;
}

} // extern "C"
