// Host build of paper_1905_05727_b200/csrc/nmsdt_math.cuh (its HOST_SEED branch emulates the 20-bit MUFU seeds), so that the
// table / polynomial logic of the fused kernels' elementary functions can be checked without a GPU.
// Built by tests/test_math_host.py:  g++ -O2 -ffp-contract=off -shared -fPIC -I<cuda>/include
#include <string.h>
#include "../paper_1905_05727_b200/csrc/nmsdt_math.cuh"

using namespace nmsdt;

extern "C" int math_probe(int fn, const double* x, int n, double a, double b, double* y0, double* y1)
{
    static double tab[MATH_TAB_DOUBLES_LOG];
    static double fa = 0.0, fb = 0.0;
    static PowCoef pw;
    if (fa != a || fb != b || fa == 0.0) {          // the power tables are built for one pair of exponents
        const double ta = a != 0.0 ? a : 4.53, tb = b != 0.0 ? b : 1.42;
        fill_math_tables(tab, ta, tb); fill_pow_coef(pw, ta, tb); fa = a; fb = b;
    }
    for (int i = 0; i < n; ++i) {
        double r0 = 0.0, r1 = 0.0;
        const double v = x[i];
        switch (fn) {
        case 0: r0 = q_rcp(v); break;
        case 1: r0 = q_sqrt(v); break;
        case 2: r0 = q_log(tab, v); break;
        case 3: q_pow_pair(tab, v, a * LOG2E, b * LOG2E, r0, r1); break;
        case 4: r0 = q_exp_neg(tab, v); break;
        case 5: r0 = floor1(v); r1 = clamp01(v); break;
        case 6: r0 = nonneg(v); r1 = cap690(v); break;
        case 8: r0 = q_sqrt_ratio_floor1(v, a); r1 = q_sqrt_ratio_floor1(a, v); break;
        case 7: if (!q_pow_tab(tab, pw, v, r0, r1)) { r0 = pow(v, pw.C); r1 = pow(v, pw.D); } break;
        default: return -1;
        }
        y0[i] = r0; y1[i] = r1;
    }
    return 0;
}
