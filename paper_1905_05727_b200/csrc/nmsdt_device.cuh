// nmsdt_device.cuh -- device-side model arithmetic of libnmsdt.so (fp64, sm_100a).
// EOS / closure (Eq. 2-5), primitive recovery (O3), Hancock predictor + limiter (O4.1-2),
// HLLC with Davis speeds (O4.3-5), Arrhenius RK4 source (Eq. 6, O5).  Readings R* are listed in DESIGN.md.
// This file shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "nmsdt_math.cuh"

namespace nmsdt {

constexpr int NGX = 16;   // left pad in doubles: interior column 0 is 128-byte aligned
constexpr int NGY = 2;    // ghost rows per side
constexpr int NG = 2;     // stencil radius

struct Params {
    int nx, ny, pitch, rows;
    long long fstride;           // doubles between planes
    double dx, dy, cfl, hmin;
    int bc_xlo, bc_xhi, bc_ylo, bc_yhi, limiter;
    // EOS (Tables I-II) and derived constants
    double gamma1, G1, iG1, cv1;
    double G2, iG2, G2p1, A, B, C, D, rho02, irho02, cv2, Tref2;
    double kA, kB, AC, BD;       // -A/(1-C), B/(1-D), A*C, B*D
    double z_min, z_max;
    // kinetics (Table III) + sub-step rule
    double Ta, Cpre, Q, theta0;
    int reactive, max_substeps;
    // fused path (nmsdt_fused.cu): C log2(e), D log2(e), 1/(Gamma2 cv2), device copy of the nmsdt_math.cuh tables
    double C2, D2, iG2cv2;
    double g1iG1;                // gamma1/(gamma1-1)
    double E1, E2, E3, R1, R2;   // Eq. 3-4 folded into the closure: see face_fast / prim_cell
    PowCoef pw;                  // exponents C, D of Eq. 3-4 and their binomial coefficients (q_pow_tab)
    const double* tab;
    const double* inflow;        // [7][ny] left boundary column captured by sim_init* (SIM_BC_INFLOW_FIXED)
};

// device-resident control block: the time step never visits the host inside sim_step
struct Ctl {
    double dt;                    // step to take next
    double tsafe;                 // T2 bound below which the R13 rule gives n_sub = 1 for tau = dt/2 (must follow dt)
    double t;
    double dt_last;
    double dt_fixed;              // > 0: sim_step_dt mode
    long long step;
    unsigned long long smax_bits; // max wavespeed of the current state, as ordered bits of a non-negative double
    int bad;
    int redo;                     // fused path: warp segments repeated with the exact rules since sim_init (R13 / R17 / power tables)
    unsigned int ticket;          // fused path: blocks of the running pass-2 sweep that have finished (the last one ends the step)
    int pad;
};

// Programmatic dependent launch (the step's kernels are chained with it, nmsdt_capi.cu): a kernel lets the next one in the
// stream be scheduled as its own blocks drain, and waits for the previous one to have completed (memory visible) before
// it touches the state or the control block.  Everything before pdl_wait() -- table copy to shared memory, barrier
// initialisation -- overlaps the predecessor's tail.  Every kernel of the chain calls pdl_wait(), so completion stays
// transitive.  Both are no-ops in a kernel that was launched without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ double clampd(double x, double lo, double hi) { return x < lo ? lo : (x > hi ? hi : x); }

// x^C and x^D from one logarithm
struct RefCurve { double x, xC, xD; };
__device__ __forceinline__ RefCurve ref_curve(const Params& P, double rho2)
{
    RefCurve r;
    r.x = rho2 * P.irho02;
    double L = log(r.x);
    r.xC = exp(P.C * L);
    r.xD = exp(P.D * L);
    return r;
}
__device__ __forceinline__ double pref2(const Params& P, const RefCurve& r) { return P.A * r.xC - P.B * r.xD; }      // Eq. 3
__device__ __forceinline__ double rho_eref2(const Params& P, const RefCurve& r)                                       // rho2 * Eq. 4
{ return P.kA * (r.xC - r.x) + P.kB * (r.xD - r.x); }

struct Prim {           // W = (rho1, rho2, un, ut, p, z1, lambda) with un the velocity normal to the sweep faces
    double r1, r2, un, ut, p, z1, lam;
};

// O3: conserved (normal/tangential momentum already ordered) -> primitives, mixture rho, floored c^2, T2
__device__ __forceinline__ void cons_to_prim(const Params& P, const double q[7], Prim& W, double& rho, double& c2, double* T2)
{
    rho = q[0] + q[1];
    double irho = 1.0 / rho;
    W.un = q[2] * irho;
    W.ut = q[3] * irho;
    double z1 = clampd(q[5], P.z_min, P.z_max);
    double z2 = 1.0 - z1;
    W.z1 = z1;
    W.r1 = q[0] / z1;
    W.r2 = q[1] / z2;
    double rhoe = q[4] - 0.5 * (q[2] * q[2] + q[3] * q[3]) * irho;
    RefCurve r = ref_curve(P, W.r2);
    double pr = pref2(P, r);
    double xi = z1 * P.iG1 + z2 * P.iG2;
    double ixi = 1.0 / xi;
    W.p = (rhoe - z2 * (rho_eref2(P, r) - pr * P.iG2)) * ixi;
    W.lam = clampd(q[6] / q[1], 0.0, 1.0);
    double r2c22 = (P.AC * r.xC - P.BD * r.xD) + P.G2p1 * (W.p - pr);
    double rc2 = (z1 * P.gamma1 * W.p * P.iG1 + z2 * r2c22 * P.iG2) * ixi;     // R10
    c2 = fmax(rc2 * irho, 1.0);
    if (T2) *T2 = P.Tref2 + (W.p - pr) / (W.r2 * P.G2 * P.cv2);                // Eq. 5
}

// one side of a face: primitives + what HLLC needs from the EOS
struct Face {
    double r1, r2, un, ut, p, z1, lam;
    double rho, rhoE, c;
};

__device__ __forceinline__ void face_state(const Params& P, const double W[7], Face& f)
{
    double z1 = W[5], z2 = 1.0 - z1;
    f.r1 = W[0]; f.r2 = W[1]; f.un = W[2]; f.ut = W[3]; f.p = W[4]; f.z1 = z1; f.lam = W[6];
    f.rho = z1 * W[0] + z2 * W[1];
    RefCurve r = ref_curve(P, W[1]);
    double pr = pref2(P, r);
    f.rhoE = z1 * W[4] * P.iG1 + z2 * (rho_eref2(P, r) + (W[4] - pr) * P.iG2) + 0.5 * f.rho * (W[2] * W[2] + W[3] * W[3]);
    double xi = z1 * P.iG1 + z2 * P.iG2;
    double r2c22 = (P.AC * r.xC - P.BD * r.xD) + P.G2p1 * (W[4] - pr);
    double rc2 = (z1 * P.gamma1 * W[4] * P.iG1 + z2 * r2c22 * P.iG2) / xi;
    f.c = sqrt(fmax(rc2 / f.rho, 1.0));
}

__device__ __forceinline__ double limited(int kind, double a, double b)
{
    double ab = a * b;
    if (kind == 0) {                                  // minmod
        double m = fabs(a) < fabs(b) ? a : b;
        return ab > 0.0 ? m : 0.0;
    }
    double m = fmin(fmin(2.0 * fabs(a), 2.0 * fabs(b)), 0.5 * fabs(a + b));   // monotonised central
    m = a > 0.0 ? m : -m;
    return ab > 0.0 ? m : 0.0;
}

// O4.1-2: limited slopes + Hancock predictor for the centre cell; returns false when the fallback fired
__device__ __forceinline__ void reconstruct(const Params& P, const Prim& Wm, const Prim& W0, const Prim& Wp, double rho0, double c20,
                                            double khalf, double WL[7], double WR[7])
{
    const double w0[7] = {W0.r1, W0.r2, W0.un, W0.ut, W0.p, W0.z1, W0.lam};
    const double wm[7] = {Wm.r1, Wm.r2, Wm.un, Wm.ut, Wm.p, Wm.z1, Wm.lam};
    const double wp[7] = {Wp.r1, Wp.r2, Wp.un, Wp.ut, Wp.p, Wp.z1, Wp.lam};
    double D[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) D[k] = limited(P.limiter, w0[k] - wm[k], wp[k] - w0[k]);
    double u = W0.un;
    double d[7];
    d[0] = u * D[0] + W0.r1 * D[2];
    d[1] = u * D[1] + W0.r2 * D[2];
    d[2] = u * D[2] + D[4] / rho0;
    d[3] = u * D[3];
    d[4] = u * D[4] + rho0 * c20 * D[2];
    d[5] = u * D[5];
    d[6] = u * D[6];
#pragma unroll
    for (int k = 0; k < 7; ++k) {
        WL[k] = w0[k] - 0.5 * D[k] - khalf * d[k];
        WR[k] = w0[k] + 0.5 * D[k] - khalf * d[k];
    }
    bool ok = (WL[0] > 0.0) && (WL[1] > 0.0) && (WR[0] > 0.0) && (WR[1] > 0.0);     // R17
    if (!ok) {
#pragma unroll
        for (int k = 0; k < 7; ++k) { WL[k] = w0[k]; WR[k] = w0[k]; }
    }
}

// O4.4-5: HLLC flux F[0..6] (component 2 = normal momentum) and face velocity
__device__ __forceinline__ void hllc(const Face& L, const Face& R, double F[7], double& uface)
{
    double SL = fmin(L.un - L.c, R.un - R.c);          // R9: Davis
    double SR = fmax(L.un + L.c, R.un + R.c);
    double mL = L.rho * (SL - L.un), mR = R.rho * (SR - R.un);
    double Sstar = (R.p - L.p + L.un * mL - R.un * mR) / (mL - mR);
    bool useL = (SL >= 0.0) || ((SR > 0.0) && (Sstar >= 0.0));
    bool star = (SL < 0.0) && (SR > 0.0);
    // selected side
    double r1 = useL ? L.r1 : R.r1, r2 = useL ? L.r2 : R.r2, un = useL ? L.un : R.un, ut = useL ? L.ut : R.ut;
    double p = useL ? L.p : R.p, z1 = useL ? L.z1 : R.z1, lam = useL ? L.lam : R.lam;
    double rho = useL ? L.rho : R.rho, rhoE = useL ? L.rhoE : R.rhoE, SK = useL ? SL : SR;
    double U[7], FK[7];
    U[0] = z1 * r1; U[1] = (1.0 - z1) * r2; U[2] = rho * un; U[3] = rho * ut; U[4] = rhoE; U[5] = z1; U[6] = U[1] * lam;
    FK[0] = U[0] * un; FK[1] = U[1] * un; FK[2] = rho * un * un + p; FK[3] = rho * un * ut; FK[4] = (rhoE + p) * un;
    FK[5] = z1 * un; FK[6] = U[6] * un;
    double chi = (SK - un) / (SK - Sstar);
    double Us[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) Us[k] = chi * U[k];
    Us[2] = rho * chi * Sstar;
    double EK = rhoE / rho;
    Us[4] = rho * chi * (EK + (Sstar - un) * (Sstar + p / (rho * (SK - un))));
#pragma unroll
    for (int k = 0; k < 7; ++k) F[k] = star ? FK[k] + SK * (Us[k] - U[k]) : FK[k];
    uface = star ? un + SK * (chi - 1.0) : un;
}

// O5: Arrhenius source over tau on one cell (conserved q, any momentum order). Updates q[4], q[6].
// p_out/c2 are not needed by callers of the unfused path.
__device__ __forceinline__ void source_cell(const Params& P, double q[7], double tau)
{
    Prim W; double rho, c2, T0;
    cons_to_prim(P, q, W, rho, c2, &T0);
    double z1 = W.z1, z2 = 1.0 - z1, lam0 = W.lam;
    double xi = z1 * P.iG1 + z2 * P.iG2;
    double beta = z2 * P.Q / (xi * P.G2 * P.cv2);
    double Tub = T0 + beta * lam0;
    int nsub = 1;
    if (Tub > 0.0) {   // R13: decision from exactly rounded operations only (no FMA contraction)
        double y = __ddiv_rn(P.Ta, Tub);
        double y2 = __dmul_rn(y, y);
        double den = __dadd_rn(__dadd_rn(__dadd_rn(1.0, y), __ddiv_rn(y2, 2.0)), __ddiv_rn(__dmul_rn(y2, y), 6.0));
        double g = __ddiv_rn(1.0, den);
        double theta = __dmul_rn(__dmul_rn(tau, P.Cpre), g);
        double r = floor(__ddiv_rn(theta, P.theta0));
        nsub = (r >= (double)(P.max_substeps - 1)) ? P.max_substeps : 1 + (int)r;
    }
    double h = tau / (double)nsub;
    double lam = lam0;
    for (int s = 0; s < nsub; ++s) {
        double k1, k2, k3, k4, T, l;
        l = lam;                 T = T0 + beta * (lam0 - l); k1 = T > 0.0 ? -l * P.Cpre * exp(-P.Ta / T) : 0.0;
        l = lam + 0.5 * h * k1;  T = T0 + beta * (lam0 - l); k2 = T > 0.0 ? -l * P.Cpre * exp(-P.Ta / T) : 0.0;
        l = lam + 0.5 * h * k2;  T = T0 + beta * (lam0 - l); k3 = T > 0.0 ? -l * P.Cpre * exp(-P.Ta / T) : 0.0;
        l = lam + h * k3;        T = T0 + beta * (lam0 - l); k4 = T > 0.0 ? -l * P.Cpre * exp(-P.Ta / T) : 0.0;
        lam = lam + h / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4);
    }
    double lam1 = clampd(lam, 0.0, lam0);
    q[6] = q[1] * lam1;
    q[4] = q[4] + q[1] * P.Q * (lam0 - lam1);
}

// order-preserving encoding of non-negative doubles for atomicMax
__device__ __forceinline__ unsigned long long dbits(double x) { return (unsigned long long)__double_as_longlong(x); }

} // namespace nmsdt
