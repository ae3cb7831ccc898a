// dt_kernel.cu -- CFL max-signal-speed reduction (a8, reading R8):
//     dt = cfl / max_{zones, active d} ( (|v_d| + c_f,d) * (1/dx_d) )
// This translation unit is compiled with -fmad=false and evaluates the per-zone expression in the
// order DESIGN.md fixes (R15), so that for identical input the dt is bit-identical to an IEEE
// evaluation without contraction.  The max itself is exact and order independent: warp shuffle ->
// block shared memory -> atomicMax on the bit pattern (all candidates are positive doubles, for
// which the IEEE ordering equals the unsigned integer ordering of the bits).
#include "grid.h"
#include <cuda_runtime.h>

namespace pluto {

__global__ void __launch_bounds__(256)
k_dtmax(Grid g, const double *__restrict__ U, StepParams *P)
{
    const long long nzone = (long long)g.n[0] * g.n[1] * g.n[2];
    double smax = 0.0;
    int bad = 0;
    for (long long z = blockIdx.x * (long long)blockDim.x + threadIdx.x; z < nzone;
         z += (long long)gridDim.x * blockDim.x) {
        int i = (int)(z % g.n[0]);
        int j = (int)((z / g.n[0]) % g.n[1]);
        int k = (int)(z / ((long long)g.n[0] * g.n[1]));
        long long c = g.at(i, j, k);
        double rho = U[c], mx = U[g.sa + c], my = U[2 * g.sa + c], mz = U[3 * g.sa + c];
        double E = U[4 * g.sa + c];
        // cell-centred B = mean of the two faces (R7); 2D: the third magnetic array is the cell B_z
        const double *b = U + S_B * g.sa;
        double B[3] = { 0.5 * (b[c] + b[g.at(i + 1 == g.n[0] ? 0 : i + 1, j, k)]),
                        0.5 * (b[g.sa + c] + b[g.sa + g.at(i, j + 1 == g.n[1] ? 0 : j + 1, k)]),
                        g.act[2] ? 0.5 * (b[2 * g.sa + c] + b[2 * g.sa + g.at(i, j, k + 1 == g.n[2] ? 0 : k + 1)])
                                 : b[2 * g.sa + c] };
        // Cheap upper bound first: c_f,d <= sqrt(a^2 + b^2) for every d, so
        //     sig_d <= (|m_d|/rho + sqrt((gamma p + B^2)/rho)) / dx_d .
        // A zone whose bound (with a 1e-9 margin for rounding) is below the thread's running
        // maximum cannot raise it and skips the exact evaluation; the maximum found is unchanged.
        {
            double ir = 1.0 / rho;
            double B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
            double pb = (g.gamma - 1.0) * (E - 0.5 * (mx * mx + my * my + mz * mz) * ir - 0.5 * B2);
            bad |= !(rho > 0.0) || !(pb > 0.0) || isinf(rho) || isinf(pb);
            double cb = sqrt((g.gamma * pb + B2) * ir);
            double bound = 0.0;
            if (g.act[0]) bound = fmax(bound, (fabs(mx) * ir + cb) * g.idx[0]);
            if (g.act[1]) bound = fmax(bound, (fabs(my) * ir + cb) * g.idx[1]);
            if (g.act[2]) bound = fmax(bound, (fabs(mz) * ir + cb) * g.idx[2]);
            if (bound * (1.0 + 1e-9) < smax) continue;     // NaN or inf: falls through to the exact path
        }
        double v[3] = { mx / rho, my / rho, mz / rho };
        double p = (g.gamma - 1.0) * (E - 0.5 * (mx * v[0] + my * v[1] + mz * v[2])
                                        - 0.5 * (B[0] * B[0] + B[1] * B[1] + B[2] * B[2]));
        if (!(rho > 0.0) || !(p > 0.0) || isinf(rho) || isinf(p)) bad = 1;
        double a2 = g.gamma * p / rho;
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
    }
    // warp max
    for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    __shared__ double wmax[8];
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = smax;
    __syncthreads();
    if (threadIdx.x < 32) {
        double m = threadIdx.x < (blockDim.x >> 5) ? wmax[threadIdx.x] : 0.0;
        for (int o = 4; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0) atomicMax(&P->smax_bits, (unsigned long long)__double_as_longlong(m));
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
}

__global__ void k_advance_time(StepParams *P) { P->time += P->dt; }

void launch_dtmax(const Grid &g, const double *U, StepParams *P, int nblocks, cudaStream_t s)
{
    k_dtmax<<<nblocks, 256, 0, s>>>(g, U, P);
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
