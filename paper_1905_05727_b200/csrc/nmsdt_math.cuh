// nmsdt_math.cuh -- branch-free fp64 elementary functions for the fused kernels of libnmsdt.so (sm_100a).
//
// The step is bound by the FP64 pipe and by issue slots: the CUDA library's div / sqrt / log /
// exp cost ~10 / ~12 / ~35 / ~28 FP64-pipe instructions each plus a slow-path test.  Every operand on this path
// is a positive normal number (densities, volume fractions, wave-speed differences, temperatures), so the
// special-case handling is dropped and the functions are rebuilt from the MUFU seeds (rcp.approx / rsqrt.approx,
// ~20 bits) + Newton steps and from two small tables held in shared memory:
//   q_rcp   1 MUFU + 3 DFMA          (<= 1 ulp for normal x)
//   q_sqrt  1 MUFU + 2 DMUL + 3 DFMA   (~1 ulp)
//   pow_pair(x) -> (x^C, x^D)  Eq. 3-4: one table-driven log (256 entries, degree-5 log1p) and two
//          table-driven exp2 (256 entries, degree-4), 25 FP64 instructions instead of ~90
//   exp_neg(y) = e^-y for the Arrhenius factor of Eq. 6
// Accuracy (tests/math_cases.py: on the host by tests/test_math_host.py, on the device by tests/test_gpu_math.py through
// sim_probe_math, against long-double library references): relative error <= 2e-16 for q_rcp / q_sqrt, absolute
// error <= 2e-16 max(1, |ln x|) for q_log, <= 8e-16 + 3e-16 |a ln x| for the powers x^a (1.2e-15 for rho2/rho02 in
// [0.5, 3]), <= 1e-15 for exp(-y), y <= 40.
// Compiles for the host too (HOST_SEED emulates the 20-bit seeds) so that the polynomial/table logic can be checked
// without a GPU.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace nmsdt {

constexpr int LOG_TAB_BITS = 8, LOG_TAB_N = 1 << LOG_TAB_BITS;     // (1/c_j, ln c_j) pairs
constexpr int EXP_TAB_BITS = 8, EXP_TAB_N = 1 << EXP_TAB_BITS;     // 2^(j/256)
constexpr int MATH_TAB_DOUBLES = 2 * LOG_TAB_N + EXP_TAB_N;        // 768 doubles = 6144 B of shared memory

#if defined(__CUDA_ARCH__)
#define NMSDT_HD __device__ __forceinline__
__device__ __forceinline__ double rcp_seed(double x) { double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
__device__ __forceinline__ double rsq_seed(double x) { double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
__device__ __forceinline__ double mk_double(int hi, int lo) { return __hiloint2double(hi, lo); }
__device__ __forceinline__ int hi_word(double x) { return __double2hiint(x); }
__device__ __forceinline__ int lo_word(double x) { return __double2loint(x); }
#else
#define NMSDT_HD inline
inline double mk_double(int hi, int lo) { uint64_t u = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo; double d; memcpy(&d, &u, 8); return d; }
inline int hi_word(double x) { uint64_t u; memcpy(&u, &x, 8); return (int)(u >> 32); }
inline int lo_word(double x) { uint64_t u; memcpy(&u, &x, 8); return (int)(u & 0xffffffffu); }
inline double rcp_seed(double x) { return mk_double(hi_word(1.0 / mk_double(hi_word(x), 0)), 0); }       // 20-bit input, 20-bit output
inline double rsq_seed(double x) { return mk_double(hi_word(1.0 / sqrt(mk_double(hi_word(x), 0))), 0); }
#endif

// polynomial coefficients: kept in the constant bank on the device so that DFMA reads them as c[][] operands
// (as 64-bit immediates each costs two moves per use)
#if defined(__CUDACC__)
#define NMSDT_KCONST static __constant__ double
#else
#define NMSDT_KCONST static const double
#endif
NMSDT_KCONST KC[10] = {
    0.0, 0.2, 1.0 / 3.0, 0.69314718055994530942,                                         // (unused), log1p series, ln 2
    0.0, 9.6181291076284772e-3, 5.5504108664821580e-2,                                   // (unused), ln2^4/24, ln2^3/6
    2.4022650695910071e-1, 6.9314718055994531e-1, 1.4426950408889634074};                // ln2^2/2, ln2, log2(e)

// min / max without the NaN rules of fmin / fmax (3 instructions instead of 5-6; operands here are never NaN on a
// valid state, and an invalid state is caught on the conserved variables)
NMSDT_HD double dmin_(double a, double b) { return a < b ? a : b; }
NMSDT_HD double dmax_(double a, double b) { return a > b ? a : b; }

// 1/x for positive (or negative) normal x: seed e0 ~ 2^-20, cubic step -> e0^3 < 2^-59
NMSDT_HD double q_rcp(double x)
{
    double r = rcp_seed(x);
    double e = fma(-x, r, 1.0);
    e = fma(e, e, e);
    return fma(r, e, r);
}

// sqrt(x) for positive normal x: seed y ~ (1+d)/sqrt(x), e = 1 - x y^2, sqrt(x) = x y (1-e)^(-1/2) truncated after the
// e^2 term (next term 5/16 e^3 < 3e-18 for the 2^-20 seed): 2 DMUL + 3 DFMA
NMSDT_HD double q_sqrt(double x)
{
    const double y = rsq_seed(x);
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(e, 0.375, 0.5) * e;
    return fma(t, p, t);
}

// Clamps decided on the high word (integer pipe instead of the FP64 pipe).  For finite x:
//   floor1(x)  = max(x, 1)      (x < 1, zero or negative -> 1; the signed compare sends negative x below 0x3ff00000)
//   clamp01(x) = min(max(x, 0), 1)
//   nonneg(x)  = max(x, 0)
//   cap690(y)  = min(y, 690) for the argument of exp(-y) (690 = 0x40859000_00000000 exactly)
//   is_pos(x)  = x > 0 for x that is zero, normal or infinite (a positive subnormal counts as zero)
NMSDT_HD bool is_pos(double x) { return hi_word(x) > 0; }
NMSDT_HD double floor1(double x) { return hi_word(x) >= 0x3ff00000 ? x : 1.0; }
NMSDT_HD double nonneg(double x) { return hi_word(x) < 0 ? 0.0 : x; }
NMSDT_HD double clamp01(double x) { const int h = hi_word(x); return h < 0 ? 0.0 : (h >= 0x3ff00000 ? 1.0 : x); }
NMSDT_HD double cap690(double y) { return hi_word(y) < 0x40859000 ? y : 690.0; }

// ln(x), x positive normal.  tab = shared-memory copy of the tables.  Absolute error ~1e-16 (+ 1 ulp of the result).
NMSDT_HD double q_log(const double* __restrict__ tab, double x)
{
    const int hx = hi_word(x);
    const int j = (hx >> (20 - LOG_TAB_BITS)) & (LOG_TAB_N - 1);
    const double m = mk_double((hx & 0x000fffff) | 0x3ff00000, lo_word(x));            // mantissa in [1,2)
    const double ed = mk_double(0x43300000, hx >> 20) - 4503599627371519.0;             // unbiased exponent: (2^52 + e_biased) - (2^52 + 1023)
    const double ic = tab[2 * j], lc = tab[2 * j + 1];
    const double r = fma(m, ic, -1.0);                                                 // |r| <= 2^-9: r^6/6 < 1e-17
    double p = fma(r, KC[1], -0.25);
    p = fma(p, r, KC[2]);
    p = fma(p, r, -0.5);
    p = fma(p, r * r, r);                                                              // log1p(r)
    return fma(ed, KC[3], lc + p);
}

// 2^(a*b) for |a*b| < 1000 (a*b is never rounded: the reduction uses the exact product through fma)
NMSDT_HD double q_exp2_prod(const double* __restrict__ tab, double a, double b)
{
    const double SH = 6755399441055744.0 / EXP_TAB_N;           // 1.5 * 2^52 / 256: ulp = 1/256
    const double t = fma(a, b, SH);
    const int N = lo_word(t);
    const double f = fma(a, b, -(t - SH));                      // |f| <= 1/512: (f ln2)^5/120 < 4e-17
    const double T = tab[2 * LOG_TAB_N + (N & (EXP_TAB_N - 1))];
    double p = fma(f, KC[5], KC[6]);
    p = fma(p, f, KC[7]);
    p = fma(p, f, KC[8]);
    const double v = fma(T, p * f, T);
    return mk_double(hi_word(v) + ((N >> EXP_TAB_BITS) << 20), lo_word(v));
}

constexpr double LOG2E = 1.4426950408889634074;

// (x^C, x^D) from one logarithm; C2 = C*log2(e), D2 = D*log2(e)
NMSDT_HD void q_pow_pair(const double* __restrict__ tab, double x, double C2, double D2, double& xC, double& xD)
{
    const double L = q_log(tab, x);
    xC = q_exp2_prod(tab, C2, L);
    xD = q_exp2_prod(tab, D2, L);
}

// e^(-y) for y >= 0 (flushes to ~1e-301 for y > 690)
NMSDT_HD double q_exp_neg(const double* __restrict__ tab, double y)
{
    return q_exp2_prod(tab, cap690(y), -KC[9]);
}

// host side: fill the 320-double table (long double arithmetic)
inline void fill_math_tables(double* tab)
{
    for (int j = 0; j < LOG_TAB_N; ++j) {
        const long double c = 1.0L + ((long double)j + 0.5L) / (long double)LOG_TAB_N;
        const double ic = (double)(1.0L / c);
        tab[2 * j] = ic;
        tab[2 * j + 1] = (double)(-logl((long double)ic));
    }
    for (int j = 0; j < EXP_TAB_N; ++j) tab[2 * LOG_TAB_N + j] = (double)exp2l((long double)j / (long double)EXP_TAB_N);
}

} // namespace nmsdt
