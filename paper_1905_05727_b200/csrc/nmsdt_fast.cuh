// nmsdt_fast.cuh -- the model arithmetic of the fused path (fp64, sm_100a), shared by the sweep kernels (nmsdt_fused.cu),
// the diagnostics reduction (nmsdt_init.cu) and the post-processing kernels (nmsdt_post.cu): primitive recovery with the
// mixture closure (O3; Eq. 2-5) and the Arrhenius source step (O5; Eq. 6; R13), built on the branch-free
// elementary functions of nmsdt_math.cuh.  `tab` is a shared-memory copy of Params::tab.  Shares nothing with oracle/.
#pragma once
#include "nmsdt_device.cuh"
#include "nmsdt_math.cuh"

namespace nmsdt {

namespace {

struct FCell {            // W = (rho1, rho2, un, ut, p, z1, lambda) + what the Hancock predictor needs
    double r1, r2, un, ut, p, z1, lam;
    double irho, rc2;     // 1/rho, rho c^2 (with the c >= 1 m/s floor of R10)
    double pr;            // p_ref2(rho2) of Eq. 3 (used by the diagnostics / post-processing kernels for T2, Eq. 5)
};

__device__ __forceinline__ double clampf(double x, double lo, double hi) { return dmin_(dmax_(x, lo), hi); }

// R13 exact sub-step count (only reached by cells hotter than the safe bound; same exactly-rounded sequence as k_source)
__device__ __noinline__ int nsub_exact(const Params& P, double Tub, double tau)
{
    if (!(Tub > 0.0)) return 1;
    double y = __ddiv_rn(P.Ta, Tub);
    double y2 = __dmul_rn(y, y);
    double den = __dadd_rn(__dadd_rn(__dadd_rn(1.0, y), __ddiv_rn(y2, 2.0)), __ddiv_rn(__dmul_rn(y2, y), 6.0));
    double g = __ddiv_rn(1.0, den);
    double theta = __dmul_rn(__dmul_rn(tau, P.Cpre), g);
    double r = floor(__ddiv_rn(theta, P.theta0));
    return (r >= (double)(P.max_substeps - 1)) ? P.max_substeps : 1 + (int)r;
}

// Arrhenius factor of Eq. 6 at (l, T) without its guard: l exp(-Ta/T); the rate is -C times this.  `good` reports the guard
// of O5 (T > 0, else the rate is 0) as one range test on the high word of y = Ta/T: y in [0, 690) <=> T > 0 and exp(-y) above
// ~1e-300 (the rate is taken as 0 beyond that; 690 = 0x40859000_00000000); T <= 0, T = +0 (y = inf) and NaN all fail the
// unsigned compare.
__device__ __forceinline__ double arr_factor(const Params& P, const double* __restrict__ tab, double l, double T, bool& good)
{
    const double y = P.Ta * q_rcp(T);
    good = (unsigned)hi_word(y) < 0x40859000u;
    return l * q_exp2_prod(tab, y, -KC[9]);
}

// one classic RK4 step of d(lambda)/dt = -lambda C exp(-Ta/T2(lambda)), T2 = T0 + beta (lam0 - lambda), from lam over h.
// The constant -C rides on the step (hC = -h C, stages k_i / (-C)) and T2 = Tb - beta lambda with Tb = T0 + beta lam0:
// 8 FP64 instructions fewer than the literal form, same values up to rounding.
// O5 tests T > 0 at every stage; one test decides all four.  If the first stage fails it, k1 = 0, the second stage sits at the
// same lambda and temperature and fails too, and so on: lambda is returned unchanged.  If it passes, the stage values of
// lambda never exceed lam (h C k >= 0 is subtracted), so with beta > 0 every later stage is at least as hot and passes.  (The
// trace liquid inside a collapsing cavity, compressed along with the air, does sit below its reference curve: T2 < 0 there.)
__device__ __forceinline__ double rk4_step(const Params& P, const double* __restrict__ tab, double Tb, double beta, double lam, double h)
{
    const double hC = -h * P.Cpre, nb = -beta;
    double l, k1, k2, k3, k4;
    bool good, g;
    l = lam;                       k1 = arr_factor(P, tab, l, fma(nb, l, Tb), good);
    l = fma(0.5 * hC, k1, lam);    k2 = arr_factor(P, tab, l, fma(nb, l, Tb), g);
    l = fma(0.5 * hC, k2, lam);    k3 = arr_factor(P, tab, l, fma(nb, l, Tb), g);
    l = fma(hC, k3, lam);          k4 = arr_factor(P, tab, l, fma(nb, l, Tb), g);
    const double r = fma(hC * (1.0 / 6.0), (k1 + k4) + 2.0 * (k2 + k3), lam);
    return good ? r : lam;
}

// R13 sub-stepped integration (only reached by cells hotter than the safe bound)
__device__ __noinline__ double rk4_substepped(const Params& P, const double* __restrict__ tab, double T0, double beta, double lam0, double tau)
{
    const double Tb = fma(beta, lam0, T0);
    const int nsub = nsub_exact(P, Tb, tau);
    const double h = tau / (double)nsub;
    double lam = lam0;
    for (int s = 0; s < nsub; ++s) lam = rk4_step(P, tab, Tb, beta, lam, h);
    return lam;
}

// O5: lambda after integrating over tau.
// SRC_FAST: one RK4 step, straight-line code; `hot` is raised when the temperature bound reaches Tsafe, i.e. when the
// R13 rule could ask for more than one sub-step: the caller then redoes its whole segment with SRC_EXACT.  Keeping
// this decision out of the marching loop keeps the loop body one basic block (the serial RK4 chain overlaps with
// the EOS evaluations of the faces).
// SRC_EXACT: the R13 rule, sub-stepped integration behind a warp-uniform branch.
enum { SRC_NONE = 0, SRC_FAST = 1, SRC_EXACT = 2 };
template <int SRC>
__device__ __forceinline__ double arrhenius_rk4(const Params& P, const double* __restrict__ tab, double T0, double beta, double lam0,
                                                double tau, double Tsafe, bool& hot)
{
    const double Tb = fma(beta, lam0, T0);
    double lam = rk4_step(P, tab, Tb, beta, lam0, tau);
    const bool h = Tb >= Tsafe;
    if (SRC == SRC_FAST) {
        hot |= h;
    } else {
        if (__any_sync(__activemask(), h)) {
            const double l2 = rk4_substepped(P, tab, T0, beta, lam0, tau);
            lam = h ? l2 : lam;
        }
    }
    return dmin_(nonneg(lam), lam0);
}

// (x^C, x^D) of Eq. 3-4 for x = rho2/rho02 by the table route.  x outside the binade table (never on a physical state):
// EX = false only raises `oor` (the sweeps then redo the segment with EX = true), EX = true takes the library powers
// behind a branch.
template <bool EX>
__device__ __forceinline__ void eos_pow(const Params& P, const double* __restrict__ tab, double x, double& xC, double& xD, bool& oor)
{
    const bool in = q_pow_tab(tab, P.pw, x, xC, xD);
    if (EX) {
        if (!in) { xC = pow(x, P.C); xD = pow(x, P.D); }
    } else {
        oor |= !in;
    }
}

// O3 (+ O5 when SRC): conserved (normal / tangential momentum ordered) -> primitives.  O3's clamp of z1 is an invariant of
// the stored q5 here (O4.6 clamps every updated cell; sim_init / sim_init_fields clamp what they write), not a step.
// SRC: the Arrhenius step over tau is applied to the cell; dE = energy moved into rho E, q6n = new z2 rho2 lambda.
// The kernels that apply the source are only launched for reactive runs (launch_sweep_fused), so there is no
// P.reactive test here.
template <int SRC, bool EX = true>
__device__ __forceinline__ void prim_cell(const Params& P, const double* __restrict__ tab, const double q[7], double tau, double Tsafe,
                                          FCell& W, double& dE, double& q6n, bool& hot)
{
    const double rho = q[0] + q[1];
    const double irho = q_rcp(rho);
    W.irho = irho;
    W.un = q[2] * irho;
    W.ut = q[3] * irho;
    const double z1 = q[5];          // within [z_min, 1 - z_min] for every state in HBM: clamped on store by the sweeps and by sim_init*
    const double z2 = 1.0 - z1;
    const double iq1 = q_rcp(q[1]);
    W.z1 = z1;
    W.r1 = q[0] * q_rcp(z1);
    W.r2 = q[1] * q_rcp(z2);
    const double rhoe = fma(-0.5, fma(q[2], W.un, q[3] * W.ut), q[4]);
    const double x = W.r2 * P.irho02;
    double xC, xD;
    eos_pow<EX>(P, tab, x, xC, xD, hot);
    const double pr = fma(P.A, xC, -P.B * xD);                                   // Eq. 3 (dead code unless T2 is wanted)
    // rho2 e_ref2 - p_ref2/Gamma2 = E1 x^C + E2 x^D - E3 x  (Eq. 3-4 folded, O2)
    const double gx = fma(P.E1, xC, fma(P.E2, xD, -P.E3 * x));
    const double xi = fma(z1, P.iG1, z2 * P.iG2);
    const double ixi = q_rcp(xi);
    double p = fma(-z2, gx, rhoe) * ixi;
    double lam = clamp01(q[6] * iq1);
    dE = 0.0; q6n = q[6];
    if (SRC != SRC_NONE) {
        const double T0 = P.Tref2 + (p - pr) * (z2 * iq1) * P.iG2cv2;            // Eq. 5 (1/rho2 = z2/q1)
        const double beta = z2 * P.Q * ixi * P.iG2cv2;
        const double lam1 = arrhenius_rk4<SRC>(P, tab, T0, beta, lam, tau, Tsafe, hot);
        dE = q[1] * P.Q * (lam - lam1);
        q6n = q[1] * lam1;
        p = fma(dE, ixi, p);                                                     // p is linear in rho e at frozen rho_k, z_k
        lam = lam1;
    }
    W.p = p; W.lam = lam; W.pr = pr;
    const double r2c22 = fma(P.R1, xC, fma(P.R2, xD, P.G2p1 * p));               // rho2 c2^2
    const double rc2 = fma(z1 * P.g1iG1, p, z2 * P.iG2 * r2c22) * ixi;           // R10
    W.rc2 = dmax_(rc2, rho);                                                      // c^2 >= 1
}

// Eq. 5 temperature of the liquid from the recovered primitives
__device__ __forceinline__ double cell_T2(const Params& P, const FCell& W) { return P.Tref2 + (W.p - W.pr) * q_rcp(W.r2) * P.iG2cv2; }

} // namespace

} // namespace nmsdt
