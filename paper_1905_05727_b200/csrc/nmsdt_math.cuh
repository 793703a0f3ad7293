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

constexpr int LOG_TAB_BITS = 8, LOG_TAB_N = 1 << LOG_TAB_BITS;     // c_j = 1 + (j + 1/2)/256: 1/c_j, ln c_j, c_j^C, c_j^D
constexpr int EXP_TAB_BITS = 8, EXP_TAB_N = 1 << EXP_TAB_BITS;     // 2^(j/256)
constexpr int POW_E_MIN = -8, POW_E_N = 16;                        // binades 2^-8 .. 2^7 of the table-driven powers
// table layout (doubles): [1/c_j][2^(j/256)][(c_j^C, c_j^D)][(2^(eC), 2^(eD))] | [ln c_j]
constexpr int IC_OFF = 0, EXP_OFF = LOG_TAB_N, POW_OFF = EXP_OFF + EXP_TAB_N, PE_OFF = POW_OFF + 2 * LOG_TAB_N;
constexpr int LC_OFF = PE_OFF + 2 * POW_E_N;
constexpr int MATH_TAB_DOUBLES = LC_OFF;                           // 1056 doubles = 8448 B: what the step kernels hold in shared memory
constexpr int MATH_TAB_DOUBLES_LOG = LC_OFF + LOG_TAB_N;           // + ln c_j for the kernels that call q_log (post-processing, probe)

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

// max(sqrt(n/d), 1) for d > 0 without a reciprocal: sqrt(n/d) = n rsqrt(n d), the reciprocal square root refined as in
// q_sqrt (seed y ~ (1+delta)/sqrt(x), e = 1 - x y^2, y (1 + e/2 + 3 e^2/8)): 7 FP64 instructions instead of the 9 of
// q_sqrt(n * q_rcp(d)), one MUFU instead of two.  n <= 0 (the c >= 1 m/s floor of R10 in strongly expanded liquid), NaN and
// overflow all give 1: one unsigned range test on the high word lets only results in [1, inf) through.
NMSDT_HD double q_sqrt_ratio_floor1(double n, double d)
{
    const double x = n * d;
    const double y = rsq_seed(x);
    const double t = x * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(e, 0.375, 0.5) * e;
    const double c = n * fma(y, p, y);
    return (unsigned)(hi_word(c) - 0x3ff00000) < 0x40000000u ? c : 1.0;
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

// ln(x), x positive normal.  tab = shared-memory copy of the tables INCLUDING the ln c_j part (MATH_TAB_DOUBLES_LOG).
// Absolute error ~1e-16 (+ 1 ulp of the result).
NMSDT_HD double q_log(const double* __restrict__ tab, double x)
{
    const int hx = hi_word(x);
    const int j = (hx >> (20 - LOG_TAB_BITS)) & (LOG_TAB_N - 1);
    const double m = mk_double((hx & 0x000fffff) | 0x3ff00000, lo_word(x));            // mantissa in [1,2)
    const double ed = mk_double(0x43300000, hx >> 20) - 4503599627371519.0;             // unbiased exponent: (2^52 + e_biased) - (2^52 + 1023)
    const double ic = tab[IC_OFF + j], lc = tab[LC_OFF + j];
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
    const double T = tab[EXP_OFF + (N & (EXP_TAB_N - 1))];
    double p = fma(f, KC[5], KC[6]);
    p = fma(p, f, KC[7]);
    p = fma(p, f, KC[8]);
    const double v = fma(T, p * f, T);
    return mk_double(hi_word(v) + ((N >> EXP_TAB_BITS) << 20), lo_word(v));
}

constexpr double LOG2E = 1.4426950408889634074;

// (x^C, x^D) for the two fixed exponents of Eq. 3-4 without a logarithm: x = 2^e c_j (1 + r), |r| <= 2^-9, so
//   x^C = 2^(eC) c_j^C (1 + r)^C,  (1 + r)^C = 1 + r (C + r (b2 + r (b3 + r (b4 + r b5)))),  b_k = binom(C, k)
// (next term binom(C,6) r^6 < 2e-18).  Two table products + 5 DFMA per power, 15 FP64 instructions for the pair against 25
// through q_log / q_exp2_prod, and no integer exponent surgery.  The binade table covers 2^-8 <= x < 2^8 (rho2/rho02 of
// nitromethane stays within [0.3, 3]); the return value says whether x was inside -- outside, the results are finite
// garbage and the caller must take another route (the sweeps redo the segment with the exact rules, see nmsdt_fused.cu).
// Relative error <= 3e-16 (table entries and coefficients are rounded long-double values).
struct PowCoef { double C, D, c[4], d[4]; };       // exponents and binom(C, 2..5), binom(D, 2..5)
NMSDT_HD bool q_pow_tab(const double* __restrict__ tab, const PowCoef& K, double x, double& xC, double& xD)
{
    const int hx = hi_word(x);
    const int j = (hx >> (20 - LOG_TAB_BITS)) & (LOG_TAB_N - 1);
    const int e = (hx >> 20) - (1023 + POW_E_MIN);                                      // negative for x < 2^-8, x <= 0, -NaN
    const int ei = e & (POW_E_N - 1);
    const double m = mk_double((hx & 0x000fffff) | 0x3ff00000, lo_word(x));            // mantissa in [1,2)
    const double r = fma(m, tab[IC_OFF + j], -1.0);
    const double sC = tab[POW_OFF + 2 * j] * tab[PE_OFF + 2 * ei];
    const double sD = tab[POW_OFF + 2 * j + 1] * tab[PE_OFF + 2 * ei + 1];
    double qc = fma(r, K.c[3], K.c[2]), qd = fma(r, K.d[3], K.d[2]);
    qc = fma(r, qc, K.c[1]); qd = fma(r, qd, K.d[1]);
    qc = fma(r, qc, K.c[0]); qd = fma(r, qd, K.d[0]);
    qc = fma(r, qc, K.C);    qd = fma(r, qd, K.D);
    xC = fma(sC * r, qc, sC);
    xD = fma(sD * r, qd, sD);
    return (unsigned)e < (unsigned)POW_E_N;
}

// (x^C, x^D) from one logarithm for arbitrary exponents; C2 = C*log2(e), D2 = D*log2(e).  Needs the ln c_j table.
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

// host side: fill the tables (MATH_TAB_DOUBLES_LOG doubles) and the binomial coefficients for the exponents C, D of
// Eq. 3-4 (long double arithmetic; the powers use the rounded 1/c_j so that c_j (1 + r) is the mantissa exactly)
inline void fill_math_tables(double* tab, double C, double D)
{
    for (int j = 0; j < LOG_TAB_N; ++j) {
        const long double c = 1.0L + ((long double)j + 0.5L) / (long double)LOG_TAB_N;
        const double ic = (double)(1.0L / c);
        const long double cj = 1.0L / (long double)ic;
        tab[IC_OFF + j] = ic;
        tab[LC_OFF + j] = (double)logl(cj);
        tab[POW_OFF + 2 * j] = (double)powl(cj, (long double)C);
        tab[POW_OFF + 2 * j + 1] = (double)powl(cj, (long double)D);
    }
    for (int j = 0; j < EXP_TAB_N; ++j) tab[EXP_OFF + j] = (double)exp2l((long double)j / (long double)EXP_TAB_N);
    for (int e = 0; e < POW_E_N; ++e) {
        tab[PE_OFF + 2 * e] = (double)exp2l((long double)(e + POW_E_MIN) * (long double)C);
        tab[PE_OFF + 2 * e + 1] = (double)exp2l((long double)(e + POW_E_MIN) * (long double)D);
    }
}
inline void fill_pow_coef(PowCoef& K, double C, double D)
{
    K.C = C; K.D = D;
    long double bc = (long double)C, bd = (long double)D;                // binom(a, 1)
    for (int k = 2; k <= 5; ++k) {
        bc *= ((long double)C - (k - 1)) / k; bd *= ((long double)D - (k - 1)) / k;
        K.c[k - 2] = (double)bc; K.d[k - 2] = (double)bd;
    }
}

} // namespace nmsdt
