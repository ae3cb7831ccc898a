// dt_kernel.cu -- CFL max-signal-speed reduction (a8, reading R8):
//     dt = cfl / max_{zones, active d} ( (|v_d| + c_f,d) * (1/dx_d) )
// This translation unit is compiled with -fmad=false and evaluates the per-zone expression in the
// order DESIGN.md fixes (R15), so that for identical input the dt is bit-identical to an IEEE
// evaluation without contraction.  The max itself is exact and order independent: warp shuffle ->
// block shared memory -> atomicMax on the bit pattern (all candidates are positive doubles, for
// which the IEEE ordering equals the unsigned integer ordering of the bits).
#include "grid.h"
#include "../../include/pluto.h"
#include <cuda_runtime.h>
#include <mutex>

namespace pluto {

// exact per-zone candidates, IEEE operations in the expression order DESIGN.md fixes (R15)
__device__ __forceinline__ double zone_sigma_exact(const Grid &g, double rho, double mx, double my, double mz,
                                                   double E, const double B[3], int &bad)
{
    double v[3] = { mx / rho, my / rho, mz / rho };
    double p = (g.gamma - 1.0) * (E - 0.5 * (mx * v[0] + my * v[1] + mz * v[2])
                                    - 0.5 * (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]));
    if (!(rho > 0.0) || !(p > 0.0) || isinf(rho) || isinf(p)) bad = 1;
    double a2 = g.gamma * p / rho;
    double smax = 0.0;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        if (!g.act[d]) continue;
        const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
        double b2  = (B[d] * B[d] + B[t1] * B[t1] + B[t2] * B[t2]) / rho;
        double bn2 = B[d] * B[d] / rho;
        double s = a2 + b2;
        double disc = s * s - 4.0 * a2 * bn2;
        if (disc < 0.0) disc = 0.0;
        double cf = sqrt(0.5 * (s + sqrt(disc)));
        double sig = (fabs(v[d]) + cf) * g.idx[d];
        if (sig > smax) smax = sig;
    }
    return smax;
}

// Fast arithmetic for the two filters below (explicit fma: this unit is compiled with -fmad=false).
__device__ __forceinline__ double rcp_nr(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    e = fma(e, e, e);
    return fma(y, e, y);
}
__device__ __forceinline__ double sqrt_nr(double x)      // x > 0
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double gq = x * y, h = 0.5 * y;
    double e = fma(-gq, h, 0.5);
    gq = fma(gq, e, gq); h = fma(h, e, h);
    e = fma(-gq, h, 0.5);
    return fma(gq, e, gq);
}

// The maximum is exact, but most zones never reach the IEEE evaluation.  A zone is skipped when an
// upper bound of its candidates lies below a value that is already known to be a lower bound of the
// global maximum (`thr`: the exact candidates this thread has seen and the running global maximum
// other warps have published).  Skipping never changes the result -- the zone that holds the maximum
// has every bound >= the maximum >= thr -- so the dt stays bit-identical and order independent.
//   filter 0:  whole rows, from the bound grid the last stage of the previous step left behind (an upper
//              bound of every candidate of the row's zones, kernels.cuh sigma_bound): rows that cannot
//              hold the maximum are never read
//   filter 1:  c_f,d <= sqrt(a^2 + b^2)  =>  sig_d <= (|m_d|/rho + sqrt((gamma p + B^2)/rho)) / dx_d
//   filter 2:  the candidates themselves in fast arithmetic (relative error <= 1e-8 even where the
//              discriminant cancels), with a 1e-7 margin
// One block walks whole rows (x contiguous); the running global maximum is re-read once per row.
// The upper z face of the top plane is read from the ghost plane nz of the state itself: the CT kernel
// leaves the final value there (ct_tma.cuh), so a z slab never reads its neighbour's memory here.
__global__ void __launch_bounds__(256)
k_dtmax(Grid g, const double *__restrict__ U, StepParams *P, BoundGrid bg, int cell_b)
{
    const int nrows = g.n[1] * g.n[2];
    const long long sa = g.sa;
    const double *__restrict__ b = U + S_B * sa;
    const double gm1 = g.gamma - 1.0;
    __shared__ double sbound[256];                       // filter 0: the bounds of the block's next 256 rows
    __shared__ double swmax[8];
    __shared__ int swarg[8];
    double smax = 0.0, published = 0.0, seen = 0.0;      // published, seen: uniform across the warp
    int nrow = 0;                                        // rows this warp has visited
    int bad = 0;
    // the block's rows are blockIdx.x + n * gridDim.x; they are taken 256 at a time: every thread fetches
    // the bound of one of them (one memory round trip per 256 rows instead of one per row)
    for (int chunk = blockIdx.x; chunk < nrows; chunk += 256 * gridDim.x) {
        {
            const long long myrow = chunk + (long long)threadIdx.x * gridDim.x;
            double bd = 1e300;
            if (bg.b && myrow < nrows) {
                const int k = (int)(myrow / g.n[1]), j = (int)(myrow - (long long)k * g.n[1]);
                bd = __longlong_as_double((long long)bg.b[(long long)(k / bg.bk) * bg.nbj + j / bg.bj]);
            }
            // the row with the largest bound is visited first: its exact candidates raise the running maximum
            // at once, and most other rows are then skipped unread
            double wb = myrow < nrows ? bd : -1.0;
            int wa = threadIdx.x;
            for (int o = 16; o > 0; o >>= 1) {
                const double ob = __shfl_xor_sync(0xffffffffu, wb, o);
                const int oa = __shfl_xor_sync(0xffffffffu, wa, o);
                if (ob > wb || (ob == wb && oa < wa)) { wb = ob; wa = oa; }
            }
            __syncthreads();                             // the previous chunk's bounds are no longer read
            sbound[threadIdx.x] = bd;
            if ((threadIdx.x & 31) == 0) { swmax[threadIdx.x >> 5] = wb; swarg[threadIdx.x >> 5] = wa; }
            __syncthreads();
        }
        int first = 0;
        {
            double fb = -2.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); w++)
                if (swmax[w] > fb) { fb = swmax[w]; first = swarg[w]; }
        }
        seen = __longlong_as_double((long long)*(volatile unsigned long long *)&P->smax_bits);
        for (int it = 0; it < 257; it++) {
            // visiting order: the row with the largest bound, then the others in order
            const int n = it == 0 ? first : it - 1;
            if (it > 0 && n == first) continue;
            const long long row64 = chunk + (long long)n * gridDim.x;
            if (row64 >= nrows) { if (it == 0) continue; else break; }
            if (sbound[n] < fmax(seen, published)) continue;                     // filter 0 (warp uniform)
            const int row = (int)row64;
            const int k = row / g.n[1], j = row - k * g.n[1];
            // the global running maximum is re-read on each of a warp's first eight visited rows, while it is
            // still rising fast, then every eighth row
            if (nrow < 8 || (nrow & 7) == 0) seen = __longlong_as_double((long long)*(volatile unsigned long long *)&P->smax_bits);
            const long long r0 = g.at(0, j, k);
            const long long upj = g.at(0, j + 1 == g.n[1] ? 0 : j + 1, k) - r0;
            const double *__restrict__ bzu = b + 2 * sa + r0 + g.st[2];
            double thr = fmax(smax, fmax(seen, published));
            for (int i = threadIdx.x; i < g.n[0]; i += blockDim.x) {
                const long long c = r0 + i;
                const double rho = U[c], mx = U[sa + c], my = U[2 * sa + c], mz = U[3 * sa + c], E = U[4 * sa + c];
                // cell-centred B = mean of the two faces (R7); 2D: the third magnetic array is the cell B_z
                // (cell_b: the GLM variant keeps cell-centred B in the three magnetic arrays)
                const double B[3] = { cell_b ? b[c] : 0.5 * (b[c] + b[r0 + (i + 1 == g.n[0] ? 0 : i + 1)]),
                                      cell_b ? b[sa + c] : 0.5 * (b[sa + c] + b[sa + c + upj]),
                                      (g.act[2] && !cell_b) ? 0.5 * (b[2 * sa + c] + bzu[i]) : b[2 * sa + c] };
                const double ir = rcp_nr(rho);
                const double B2 = fma(B[0], B[0], fma(B[1], B[1], B[2] * B[2]));
                const double vx = mx * ir, vy = my * ir, vz = mz * ir;
                const double pf = gm1 * (E - 0.5 * fma(mx, vx, fma(my, vy, mz * vz)) - 0.5 * B2);
                const double a2 = g.gamma * pf * ir;
                // rho <= 0, p <= 0, NaN or inf: flag, and let the exact path decide what enters the maximum
                const bool odd = (unsigned)(__double2hiint(rho) - 0x00100000) >= 0x7fe00000u ||
                                 (unsigned)(__double2hiint(pf) - 0x00100000) >= 0x7fe00000u;
                if (!odd) {
                    const double cb = sqrt_nr(fma(B2, ir, a2));
                    double ub = 0.0;
                    if (g.act[0]) ub = fmax(ub, (fabs(vx) + cb) * g.idx[0]);
                    if (g.act[1]) ub = fmax(ub, (fabs(vy) + cb) * g.idx[1]);
                    if (g.act[2]) ub = fmax(ub, (fabs(vz) + cb) * g.idx[2]);
                    if (ub * (1.0 + 1e-9) < thr) continue;                       // filter 1
                    const double v[3] = { vx, vy, vz };
                    const double s = fma(B2, ir, a2);
                    double est = 0.0;
#pragma unroll
                    for (int d = 0; d < 3; d++) {
                        if (!g.act[d]) continue;
                        const double disc = fma(s, s, -4.0 * a2 * (B[d] * B[d] * ir));
                        const double cf = sqrt_nr(0.5 * (s + sqrt_nr(fmax(disc, 1e-300))));
                        est = fmax(est, (fabs(v[d]) + cf) * g.idx[d]);
                    }
                    if (est * (1.0 + 1e-7) < thr) continue;                      // filter 2
                }
                const double sig = zone_sigma_exact(g, rho, mx, my, mz, E, B, bad);
                if (sig > smax) smax = sig;
                if (sig > thr) thr = sig;
            }
            // publish the warp's maximum when it raises the global one (rare after the first rows)
            if (nrow < 8 || (nrow & 7) == 7) {
                double wm = smax;
                for (int o = 16; o > 0; o >>= 1) wm = fmax(wm, __shfl_xor_sync(0xffffffffu, wm, o));
                if ((threadIdx.x & 31) == 0 && wm > fmax(seen, published))
                    atomicMax(&P->smax_bits, (unsigned long long)__double_as_longlong(wm));
                published = fmax(published, wm);
            }
            nrow++;
        }
    }
    {
        double wm = smax;
        for (int o = 16; o > 0; o >>= 1) wm = fmax(wm, __shfl_xor_sync(0xffffffffu, wm, o));
        if ((threadIdx.x & 31) == 0 && wm > fmax(seen, published))
            atomicMax(&P->smax_bits, (unsigned long long)__double_as_longlong(wm));
    }
    if (bad) P->err = 1;
}

// mode 0: CFL dt for the step about to start; mode 1: imposed dt; mode 2: probe only (get_dt)
__global__ void k_dtfinish(Grid g, StepParams *P, int mode)
{
    double smax = __longlong_as_double((long long)P->smax_bits);
    P->smax_bits = 0ull;
    double dt = (mode == 1) ? P->dt_fixed : g.cfl / smax;
    if (mode == 2) { P->dt_probe = dt; return; }
    P->dt = dt;
    for (int d = 0; d < 3; d++) P->dtdx[d] = dt / g.dx[d];
    // GLM variant (glm.cuh, reading R20): c_h = cfl min_d(dx_d) / dt, damping factor of psi over the step
    double h = 0.0;
    for (int d = 0; d < 3; d++) if (g.act[d] && (h == 0.0 || g.dx[d] < h)) h = g.dx[d];
    P->glm_ch = g.cfl * h / dt;
    P->glm_damp = exp(-dt * P->glm_ch / kGlmCr);
}

__global__ void k_advance_time(StepParams *P) { P->time += P->dt; }

void launch_dtmax(const Grid &g, const double *U, StepParams *P, BoundGrid bg, int cell_b, int nblocks, cudaStream_t s)
{
    k_dtmax<<<nblocks, 256, 0, s>>>(g, U, P, bg, cell_b);
}
void launch_dtfinish(const Grid &g, StepParams *P, int mode, cudaStream_t s)
{
    k_dtfinish<<<1, 1, 0, s>>>(g, P, mode);
}
void launch_advance_time(StepParams *P, cudaStream_t s) { k_advance_time<<<1, 1, 0, s>>>(P); }

} // namespace pluto

// ---------------------------------------------------------------- fp64 peak probe
// 8 independent DFMA chains per thread, no memory traffic: measures what the fp64 pipe sustains.
// (In this -fmad=false unit the FMAs are written explicitly with fma().)
namespace pluto {

__global__ void __launch_bounds__(256) k_fp64_probe(double *out, int iters, double seed)
{
    double a0 = seed + threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-6;
    for (int i = 0; i < iters; i++) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456) out[0] = r;     // never true: keeps the loop alive
}

double probe_fp64_gflops(cudaStream_t s)
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double *out = nullptr;
    if (cudaMalloc((void **)&out, 8) != cudaSuccess) return NAN;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 20000, blocks = sms * 8, threads = 256;
    k_fp64_probe<<<blocks, threads, 0, s>>>(out, 2000, 1.0);          // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(e0, s);
        k_fp64_probe<<<blocks, threads, 0, s>>>(out, iters, 1.0);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double gf = 2.0 * 8.0 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-9;
        if (gf > best) best = gf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return cudaGetLastError() == cudaSuccess ? best : NAN;
}

} // namespace pluto

// ---------------------------------------------------------------- pluto_cfl_dt_noalloc (include/pluto.h)
// The CFL reduction above, for callers that must not let this library allocate: a host application that
// hands every byte of device memory to its own pool at start-up (an AMR framework's arena, a caching
// allocator run at a high memory fraction) cannot count on a cudaMalloc inside a library succeeding, and
// one that calls from a latency-critical loop cannot afford the device-wide synchronisation that
// cudaMalloc / cudaFree imply.  pluto_init needs a context (state arrays, scalars, bound grid); this entry
// point needs none: the caller passes its own state and its own output, and the only memory in between --
// one partial maximum per row of zones plus a flag word -- lives in the file-scope array below, which is
// part of the loaded module on every device (PLUTO_NOALLOC_SCRATCH_BYTES, held until the process exits).
//
// The per-zone candidate is zone_sigma_exact() of this file, so for the same state the dt is bit-identical
// to pluto_get_dt().  There are no filters here: every zone takes the IEEE evaluation.
namespace pluto { int report_error(int code, const char *fmt, ...); }

namespace {

constexpr int kNoallocMaxRows = PLUTO_NOALLOC_MAX_ROWS;
constexpr int kNoallocHeader = 32;                         // 256 bytes in front of the row maxima: [0] = unphysical-zone flag
static_assert((kNoallocMaxRows + kNoallocHeader) * 8 == PLUTO_NOALLOC_SCRATCH_BYTES, "header and limit disagree");

// Scratch of pluto_cfl_dt_noalloc.  In HOST code this name is only a handle for cudaGetSymbolAddress (passing
// it to a kernel would hand the kernel a host address); noalloc_scratch() below resolves the device address.
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kNoallocMaxRows + kNoallocHeader];

// One warp per row of nx zones of the caller's unpadded state U[8][nz][ny][nx] (cell-centred B in U[4..6]).
// Writes the row's maximum candidate (bit pattern of a non-negative double) to scratch[header + row].
__global__ void __launch_bounds__(256)
k_rowmax_noalloc(pluto::Grid g, const double *__restrict__ U, unsigned long long *__restrict__ scratch)
{
    const int nx = g.n[0];
    const long long nrows = (long long)g.n[1] * g.n[2];
    const long long zones = nrows * nx;
    const int lane = threadIdx.x & 31;
    const long long warp0 = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long nwarps = (long long)gridDim.x * (blockDim.x >> 5);
    int bad = 0;
    for (long long row = warp0; row < nrows; row += nwarps) {
        const double *__restrict__ r = U + row * nx;
        double smax = 0.0;
        for (int i = lane; i < nx; i += 32) {
            const double B[3] = { r[4 * zones + i], r[5 * zones + i], r[6 * zones + i] };
            const double sig = pluto::zone_sigma_exact(g, r[i], r[zones + i], r[2 * zones + i], r[3 * zones + i],
                                                       r[7 * zones + i], B, bad);
            if (sig > smax) smax = sig;
        }
        for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        if (lane == 0) scratch[kNoallocHeader + row] = (unsigned long long)__double_as_longlong(smax);
    }
    if (bad) scratch[0] = 1ull;
}

// One block: the maximum of the row maxima, then out[0] = dt = cfl / max, out[1] = max, out[2] = 1.0 if a zone
// with non-positive or non-finite density / pressure was met (else 0.0).
__global__ void __launch_bounds__(1024)
k_finish_noalloc(double cfl, long long nrows, const unsigned long long *__restrict__ scratch, double *__restrict__ out)
{
    __shared__ unsigned long long sm[32];
    unsigned long long m = 0ull;                            // candidates are non-negative: bit order = value order
    for (long long r = threadIdx.x; r < nrows; r += blockDim.x) {
        const unsigned long long v = scratch[kNoallocHeader + r];
        if (v > m) m = v;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long v = __shfl_xor_sync(0xffffffffu, m, o);
        if (v > m) m = v;
    }
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); w++) if (sm[w] > m) m = sm[w];
        const double smax = __longlong_as_double((long long)m);
        out[0] = cfl / smax;
        out[1] = smax;
        out[2] = scratch[0] ? 1.0 : 0.0;
    }
}

// Device address of g_noalloc_scratch on the CURRENT device, resolved once per device ordinal.
unsigned long long *noalloc_scratch(int dev, cudaError_t &err)
{
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static unsigned long long *addr[kMaxDevices] = {};
    err = cudaSuccess;
    if (dev < 0 || dev >= kMaxDevices) { err = cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void *p = nullptr;
        err = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (err != cudaSuccess) return nullptr;
        addr[dev] = (unsigned long long *)p;
    }
    return addr[dev];
}

} // namespace

extern "C" int pluto_cfl_dt_noalloc(const double *U_dev, int nx, int ny, int nz, double Lx, double Ly, double Lz,
                                    double gamma, double cfl, double *out_dev, void *cuda_stream)
{
    using pluto::report_error;
    if (!U_dev || !out_dev) return report_error(PLUTO_EINVAL, "pluto_cfl_dt_noalloc: U_dev and out_dev must be device pointers, not NULL");
    if (nx < 2 || ny < 2 || nz < 1) return report_error(PLUTO_EINVAL, "pluto_cfl_dt_noalloc: needs nx >= 2, ny >= 2, nz >= 1");
    if (!(Lx > 0.0) || !(Ly > 0.0) || !(Lz > 0.0) || !(gamma > 1.0) || !(cfl > 0.0))
        return report_error(PLUTO_EINVAL, "pluto_cfl_dt_noalloc: box lengths and cfl must be positive, gamma > 1");
    const long long nrows = (long long)ny * nz;
    if (nrows > kNoallocMaxRows)
        return report_error(PLUTO_ENOMEM, "pluto_cfl_dt_noalloc: ny * nz = %lld rows exceed the built-in scratch of "
                            "PLUTO_NOALLOC_MAX_ROWS = %d rows (this entry point never allocates; use pluto_init / "
                            "pluto_get_dt for larger boxes)", nrows, kNoallocMaxRows);
    int dev = -1, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return report_error(PLUTO_ECUDA, "pluto_cfl_dt_noalloc: no CUDA device (%s): there is no CPU fallback", cudaGetErrorString(e));
    unsigned long long *scratch = noalloc_scratch(dev, e);
    if (!scratch) return report_error(PLUTO_ECUDA, "pluto_cfl_dt_noalloc: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) sms = 148;

    pluto::Grid g{};
    const int n[3] = { nx, ny, nz };
    const double L[3] = { Lx, Ly, Lz };
    for (int a = 0; a < 3; a++) {
        g.n[a] = n[a];
        g.act[a] = n[a] > 1;
        g.dx[a] = L[a] / n[a];                // the arithmetic of pluto_set_box, so that 1/dx agrees to the bit
        g.idx[a] = 1.0 / g.dx[a];
    }
    g.gamma = gamma;
    g.cfl = cfl;

    cudaStream_t s = (cudaStream_t)cuda_stream;
    // the flag word keeps the previous call's value: it has to start at zero (the row maxima need no clearing,
    // every row this call reads is written by this call first)
    e = cudaMemsetAsync(scratch, 0, kNoallocHeader * sizeof(unsigned long long), s);
    if (e != cudaSuccess) return report_error(PLUTO_ECUDA, "pluto_cfl_dt_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
    const long long want = (nrows + 7) / 8;                                  // 8 warps per block, one row per warp
    const int blocks = (int)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    k_rowmax_noalloc<<<blocks, 256, 0, s>>>(g, U_dev, scratch);
    k_finish_noalloc<<<1, 1024, 0, s>>>(cfl, nrows, scratch, out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return report_error(PLUTO_ECUDA, "pluto_cfl_dt_noalloc: launch: %s", cudaGetErrorString(e));
    return PLUTO_OK;
}
