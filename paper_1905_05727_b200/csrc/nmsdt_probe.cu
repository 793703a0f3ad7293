// nmsdt_probe.cu -- measurement probes (include/nmsdt_probe.h): bench.py's roofline block and the accuracy tests of the
// fused path's elementary functions call them; no call of the method (include/nmsdt.h) does.  Kept in a translation unit of
// their own so that the step kernels' sources hold the method only.
#include "nmsdt_host.h"
#include "nmsdt_math.cuh"

namespace nmsdt {

// ---------------------------------------------------------------------------------------------------------
// FP64 FMA throughput probe: 8 independent DFMA chains per thread
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_fp64(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
}

int launch_probe_fp64(cudaStream_t s, double* gflops, double* ms_out)
{
    const int blocks = 148 * 8, threads = 256, iters = 1 << 14;
    double* d = nullptr;
    if (cudaMalloc(&d, sizeof(double) * blocks * threads) != cudaSuccess) return -2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_probe_fp64<<<blocks, threads, 0, s>>>(d, 1024, 0.999999, 1e-9);   // warm-up
    float best = 1e30f;
    for (int r = 0; r < 5; ++r) {
        cudaEventRecord(e0, s);
        k_probe_fp64<<<blocks, threads, 0, s>>>(d, iters, 0.999999, 1e-9);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    if (cudaGetLastError() != cudaSuccess) return -2;
    const double flop = 2.0 * 8.0 * (double)iters * blocks * threads;
    *gflops = flop / (best * 1e-3) * 1e-9;
    *ms_out = best;
    return 0;
}

// ---------------------------------------------------------------------------------------------------------
// Issue-slot probe: 8 independent DFMA chains per thread with M independent 32-bit ALU instructions (LOP3) interleaved per
// 8 DFMA, at the sweeps' residency (4 warps per scheduler).  Answers whether the other half of the sweeps' instruction
// stream can hide under the half-rate FP64 pipe: T(M)/T(0) = 1 for M <= 8 if a DFMA holds the scheduler's issue port for
// one cycle, (16 + M)/16 if it holds it for the two cycles its 16 lanes are busy.
// ---------------------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(128) k_probe_issue(double* out, int iters, double a, double b, unsigned c)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    unsigned y[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) y[k] = threadIdx.x * 8 + k;
    // (xor and add alternate on every chain so that no two consecutive instructions of a chain fold into one)
    for (int i = 0; i < iters; i += 2) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                double& x = r == 0 ? x0 : r == 1 ? x1 : r == 2 ? x2 : r == 3 ? x3 : r == 4 ? x4 : r == 5 ? x5 : r == 6 ? x6 : x7;
                asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x) : "d"(a), "d"(b));
#pragma unroll
                for (int m = 0; m < (M + 7 - r) / 8; ++m) {          // M / 8 each, the first M % 8 DFMA one more
                    unsigned& yy = y[(r + 3 * m) & 7];
                    if ((h + m) & 1) asm volatile("add.u32 %0, %0, %1;" : "+r"(yy) : "r"(c));
                    else             asm volatile("xor.b32 %0, %0, %1;" : "+r"(yy) : "r"(c));
                }
            }
        }
    }
    unsigned ys = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) ys ^= y[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7 + (double)ys;
}

template <int M>
static float time_probe_issue(cudaStream_t s, double* d, int blocks, int iters, cudaEvent_t e0, cudaEvent_t e1)
{
    k_probe_issue<M><<<blocks, 128, 0, s>>>(d, 256, 0.999999, 1e-9, 0x5bd1e995u);      // warm-up
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        cudaEventRecord(e0, s);
        k_probe_issue<M><<<blocks, 128, 0, s>>>(d, iters, 0.999999, 1e-9, 0x5bd1e995u);
        cudaEventRecord(e1, s);
        cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    return best;
}

// ms[k] = time of the probe with M = 0, 4, 8, 16 other instructions per 8 DFMA (4 blocks of 4 warps per SM, one wave)
int launch_probe_issue(cudaStream_t s, double ms[4])
{
    int dev = 0, nsm = 148; cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int blocks = nsm * 4, iters = 1 << 13;
    double* d = nullptr;
    if (cudaMalloc(&d, sizeof(double) * blocks * 128) != cudaSuccess) return -2;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    ms[0] = time_probe_issue<0>(s, d, blocks, iters, e0, e1);
    ms[1] = time_probe_issue<4>(s, d, blocks, iters, e0, e1);
    ms[2] = time_probe_issue<8>(s, d, blocks, iters, e0, e1);
    ms[3] = time_probe_issue<16>(s, d, blocks, iters, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    return cudaGetLastError() == cudaSuccess ? 0 : -2;
}

// ---------------------------------------------------------------------------------------------------------------
// sim_probe_math: evaluate the elementary functions of nmsdt_math.cuh on device arrays (accuracy tests)
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_probe_math(const __grid_constant__ PowCoef pw, const double* __restrict__ tab_g, int fn, const double* __restrict__ x, int n, double a, double b,
                                                    double* __restrict__ y0, double* __restrict__ y1)
{
    __shared__ __align__(16) double s_tab[MATH_TAB_DOUBLES_LOG];
    for (int i = threadIdx.x; i < MATH_TAB_DOUBLES_LOG; i += blockDim.x) s_tab[i] = tab_g[i];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double v = x[i];
    double r0 = 0.0, r1 = 0.0;
    switch (fn) {
    case 0: r0 = q_rcp(v); break;
    case 1: r0 = q_sqrt(v); break;
    case 2: r0 = q_log(s_tab, v); break;
    case 3: q_pow_pair(s_tab, v, a * LOG2E, b * LOG2E, r0, r1); break;      // (v^a, v^b)
    case 4: r0 = q_exp_neg(s_tab, v); break;
    case 5: r0 = floor1(v); r1 = clamp01(v); break;
    case 6: r0 = nonneg(v); r1 = cap690(v); break;
    case 8: r0 = q_sqrt_ratio_floor1(v, a); r1 = q_sqrt_ratio_floor1(a, v); break;   // max(sqrt(x/a), 1), max(sqrt(a/x), 1)
    case 7: if (!q_pow_tab(s_tab, pw, v, r0, r1)) { r0 = pow(v, pw.C); r1 = pow(v, pw.D); } break;   // the step kernels' route for Eq. 3-4
    default: break;
    }
    y0[i] = r0; y1[i] = r1;
}

int launch_probe_math(const PowCoef& pw, const double* tab_dev, int fn, const double* host_x, int n, double a, double b, double* host_y0, double* host_y1,
                      cudaStream_t s)
{
    double *dx = nullptr, *dy = nullptr;
    if (cudaMalloc(&dx, sizeof(double) * n) != cudaSuccess) return -2;
    if (cudaMalloc(&dy, sizeof(double) * 2 * n) != cudaSuccess) { cudaFree(dx); return -2; }
    cudaMemcpyAsync(dx, host_x, sizeof(double) * n, cudaMemcpyHostToDevice, s);
    k_probe_math<<<(n + 127) / 128, 128, 0, s>>>(pw, tab_dev, fn, dx, n, a, b, dy, dy + n);
    cudaMemcpyAsync(host_y0, dy, sizeof(double) * n, cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(host_y1, dy + n, sizeof(double) * n, cudaMemcpyDeviceToHost, s);
    const cudaError_t e = cudaStreamSynchronize(s);
    cudaFree(dx); cudaFree(dy);
    return e == cudaSuccess ? 0 : -2;
}

} // namespace nmsdt
