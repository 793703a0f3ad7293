// nmsdt_fused.cu -- the production step kernels of libnmsdt.so (SIM_VARIANT_FUSED; fp64, sm_100a).
//
// One time step (O6; Strang splitting P:149) is two passes over the state:
//   pass 1 = S(dt/2) applied on load + directional sweep d1          (k_xsweep<LEAD> or k_ysweep<LEAD>)
//   pass 2 = directional sweep d2 + S(dt/2) on the updated cell + max-wavespeed partial of the new state
//                                                                     (k_xsweep<TRAIL> or k_ysweep<TRAIL>)
// and the block of pass 2 that finishes last ends the step (t += dt, next CFL dt: step_end_by_last_block; the one-thread k_ctl
// is launched only by the piecewise slab calls).  Algorithmic HBM traffic: 2 x (7 read + 7 written) planes = 224 B per cell-step.  The arithmetic is that of nmsdt_device.cuh (O3-O5) with the branch-free elementary
// functions of nmsdt_math.cuh; a warp whose segment holds a cell that needs one of the rare rules (RK4 sub-steps R13,
// first-order fallback R17, a density outside the power tables) repeats the segment with the exact rules.
//
//   k_ysweep: a thread owns a column and marches along y; a warp's next input row (32 columns x 7 planes) is staged by
//             one bulk tensor copy (TMA, mbarrier-signalled) two rows ahead; the primitive window and the previous
//             right-face state live in thread-private shared-memory slots (value pairs, 128-bit accesses), the
//             half-finished update of the previous cell in registers; every load/store is a coalesced 256-byte row piece
//             and nothing is recomputed (4 ramp-up rows per segment).
//   k_xsweep: a warp owns a row segment and marches along x in chunks of 64 cells, 2 adjacent cells per lane
//             (128-bit loads/stores).  Neighbour primitives, the right-face state and the face flux cross lanes through
//             three 33-slot rings of value pairs in shared memory (slot = lane counter mod 33, so lane 31's entry of the previous
//             chunk is lane 0's left neighbour: no halo recomputation, no copies); 3 __syncwarp per chunk.
#include <type_traits>
#include <cuda.h>           // CUtensorMap (type only: the encoder is fetched from the driver at run time, nmsdt_capi.cu)
#include "nmsdt_host.h"
#include "nmsdt_fast.cuh"

namespace nmsdt {

namespace {

// pass kinds: PLAIN = sweep only; LEAD = S(dt/2) on load + sweep; TRAIL = sweep + S(dt/2) + wavespeed of the new state;
// TRAIL_INERT = sweep + wavespeed (inert runs: pass 1 is PLAIN, pass 2 is TRAIL_INERT)
enum { MODE_PLAIN = 0, MODE_LEAD = 1, MODE_TRAIL = 2, MODE_TRAIL_INERT = 3 };

// A face state: the reconstructed primitives, the mixture density and sound speed -- what both sides of a face need for the wave
// speeds -- and either the total energy or (x^C, x^D) of its liquid density.  Only the side the HLLC fan selects needs the total
// energy, so with DEFER hllc_fast forms it after the selection from (x^C, x^D): 11 FP64 instructions per face state become 12
// per face (-10 per cell and pass).  The price is a longer dependency chain inside the flux; every sweep kernel takes it
// (-1.8 ... -2.8 % each) except k_xsweep<TRAIL>, which runs 12 warps per SM with its trailing source chains already latency
// bound and got 1.1 % slower with it: that one forms the energy with the face state as before.
struct FFace { double r1, r2, un, ut, p, z1, lam, rho, c, rhoE, xC, xD; };

// E(rho1, rho2, z1, p) + kinetic energy (O4.3): Eq. 3-4 enter through (p - p_ref2)/Gamma2 + rho2 e_ref2 = p/Gamma2 + E1 x^C + E2 x^D - E3 x
__device__ __forceinline__ double face_energy(const Params& P, double r2, double un, double ut, double p, double z1, double rho, double xC, double xD)
{
    const double brk = fma(p, P.iG2, fma(P.E1, xC, fma(P.E2, xD, -P.E3 * (r2 * P.irho02))));
    const double kin = 0.5 * rho * fma(un, un, ut * ut);
    return fma(z1 * P.iG1, p, fma(1.0 - z1, brk, kin));
}

template <bool EX, bool DEFER>
__device__ __forceinline__ void face_fast(const Params& P, const double* __restrict__ tab, const double W[7], FFace& f, bool& oor)
{
    const double z1 = W[5], z2 = 1.0 - z1, p = W[4];
    f.r1 = W[0]; f.r2 = W[1]; f.un = W[2]; f.ut = W[3]; f.p = p; f.z1 = z1; f.lam = W[6];
    const double rho = fma(z1, W[0], z2 * W[1]);
    f.rho = rho;
    const double x = W[1] * P.irho02;
    double xC, xD;
    eos_pow<EX>(P, tab, x, xC, xD, oor);
    f.xC = xC; f.xD = xD;
    f.rhoE = DEFER ? 0.0 : face_energy(P, W[1], W[2], W[3], p, z1, rho, xC, xD);
    // Eq. 3-4 enter the sound speed through rho2 c2^2 = (Gamma2+1) p + R1 x^C + R2 x^D (O2)
    const double xi = fma(z1, P.iG1, z2 * P.iG2);
    const double r2c22 = fma(P.R1, xC, fma(P.R2, xD, P.G2p1 * p));
    const double rc2 = fma(z1 * P.g1iG1, p, z2 * P.iG2 * r2c22);
    f.c = q_sqrt_ratio_floor1(rc2, xi * rho);            // c = sqrt(max(rho c^2 / rho, 1)) (R10)
}

template <int LIM>
__device__ __forceinline__ double limited_f(double a, double b)
{
    if (LIM == 0) {                                                               // minmod (R5)
        // a b > 0 <=> equal sign bits and both non-zero; if either is zero the smaller magnitude is that zero
        const double m = fabs(a) < fabs(b) ? a : b;
        return ((__double2hiint(a) ^ __double2hiint(b)) >= 0) ? m : 0.0;
    }
    double m = dmin_(dmin_(2.0 * fabs(a), 2.0 * fabs(b)), 0.5 * fabs(a + b));     // monotonised central
    m = a > 0.0 ? m : -m;
    return a * b > 0.0 ? m : 0.0;
}

// O4.1-2 for the centre cell W0, given the one-sided differences a = W0 - W(-1), b = W(+1) - W0.
// R17 first-order fallback (a predicted face density <= 0 -> WL = WR = W0).  It never fires at CFL 0.4 (nor at 10x that
// step), so the marching loop does not carry it: EXACT = false only raises `redo` for such a cell, and the caller
// repeats the warp's whole segment with EXACT = true (the pass is out of place), where the fallback is applied without a
// branch: the four densities are predicted first; if one of them is not positive they are replaced by the cell values
// and the other five slopes are zeroed, which makes their face values equal the cell values exactly
// (fma(+-0.5, 0, fma(-k, 0, w)) = w).
template <int LIM, bool EXACT>
__device__ __forceinline__ void recon_core(const Params& P, const FCell& W0, const double a[7], const double b[7], double khalf, double WL[7],
                                           double WR[7], bool counted, bool& redo)
{
    const double w0[7] = {W0.r1, W0.r2, W0.un, W0.ut, W0.p, W0.z1, W0.lam};
    double D[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) D[k] = limited_f<LIM>(a[k], b[k]);
    // predictor W - k (u D + coupling terms) (O4.2), written so that every component is a chain of fma on k u, k D_u, k D_p
    const double ku = khalf * W0.un;
    const double kDu = khalf * D[2];
    const double m0 = fma(-ku, D[0], fma(-kDu, W0.r1, w0[0]));
    const double m1 = fma(-ku, D[1], fma(-kDu, W0.r2, w0[1]));
    WL[0] = fma(-0.5, D[0], m0); WR[0] = fma(0.5, D[0], m0);
    WL[1] = fma(-0.5, D[1], m1); WR[1] = fma(0.5, D[1], m1);
    // all four > 0 (a positive subnormal counts as zero)
    const bool ok = min(min(hi_word(WL[0]), hi_word(WL[1])), min(hi_word(WR[0]), hi_word(WR[1]))) > 0;
    if (EXACT) {
        WL[0] = ok ? WL[0] : w0[0]; WR[0] = ok ? WR[0] : w0[0];
        WL[1] = ok ? WL[1] : w0[1]; WR[1] = ok ? WR[1] : w0[1];
#pragma unroll
        for (int k = 2; k < 7; ++k) D[k] = ok ? D[k] : 0.0;
    } else {
        redo |= counted && !ok;
    }
    // (EXACT with a fallback cell: every D[k] is zero from here on and the densities above were replaced, so k Du = 0 too)
    const double kDu2 = khalf * D[2], kDp = khalf * D[4];
    double m[7];
    m[2] = fma(-ku, D[2], fma(-kDp, W0.irho, w0[2]));
    m[3] = fma(-ku, D[3], w0[3]);
    m[4] = fma(-ku, D[4], fma(-kDu2, W0.rc2, w0[4]));
    m[5] = fma(-ku, D[5], w0[5]);
    m[6] = fma(-ku, D[6], w0[6]);
#pragma unroll
    for (int k = 2; k < 7; ++k) {
        WL[k] = fma(-0.5, D[k], m[k]);
        WR[k] = fma(0.5, D[k], m[k]);
    }
}

template <int LIM, bool EXACT>
__device__ __forceinline__ void recon_fast(const Params& P, const FCell& Wm, const FCell& W0, const FCell& Wp, double khalf, double WL[7],
                                           double WR[7], bool counted, bool& redo)
{
    const double a[7] = {W0.r1 - Wm.r1, W0.r2 - Wm.r2, W0.un - Wm.un, W0.ut - Wm.ut, W0.p - Wm.p, W0.z1 - Wm.z1, W0.lam - Wm.lam};
    const double b[7] = {Wp.r1 - W0.r1, Wp.r2 - W0.r2, Wp.un - W0.un, Wp.ut - W0.ut, Wp.p - W0.p, Wp.z1 - W0.z1, Wp.lam - W0.lam};
    recon_core<LIM, EXACT>(P, W0, a, b, khalf, WL, WR, counted, redo);
}

// O4.4-5: HLLC flux F[0..6] (component 2 = normal momentum), F[7] = face velocity
template <bool DEFER>
__device__ __forceinline__ void hllc_fast(const Params& P, const FFace& L, const FFace& R, double F[8])
{
    const double SL = dmin_(L.un - L.c, R.un - R.c);                  // R9: Davis
    const double SR = dmax_(L.un + L.c, R.un + R.c);
    const double mL = L.rho * (SL - L.un), mR = R.rho * (SR - R.un);
    const double Sstar = (R.p - L.p + fma(L.un, mL, -R.un * mR)) * q_rcp(mL - mR);
    // sign tests on the high words (integer pipe).  They differ from the floating-point comparisons only for -0.0 and
    // subnormals: SL = -0.0 enters the star branch with SKs = -0.0, where F* = F_L exactly; S* = -0.0 takes the right
    // star state, whose flux equals the left one at S* = 0 (F*_L - F*_R = S* (U*_L - U*_R)); a subnormal SR counts as 0.
    const bool sl_neg = hi_word(SL) < 0, sr_pos = hi_word(SR) > 0;
    const bool useL = !sl_neg || (sr_pos && hi_word(Sstar) >= 0);
    const bool star = sl_neg && sr_pos;
    const double r1 = useL ? L.r1 : R.r1, r2 = useL ? L.r2 : R.r2, un = useL ? L.un : R.un, ut = useL ? L.ut : R.ut;
    const double p = useL ? L.p : R.p, z1 = useL ? L.z1 : R.z1, lam = useL ? L.lam : R.lam;
    const double rho = useL ? L.rho : R.rho, SK = useL ? SL : SR;
    double rhoE;                                                       // total energy of the selected side
    if (DEFER) rhoE = face_energy(P, r2, un, ut, p, z1, rho, useL ? L.xC : R.xC, useL ? L.xD : R.xD);
    else rhoE = useL ? L.rhoE : R.rhoE;
    // chi = (SK-un)/(SK-S*) and p/(SK-un) from one reciprocal; outside the fan SKs = 0 and the star terms vanish
    const double a = SK - un, b = SK - Sstar;
    const double rab = star ? q_rcp(a * b) : 0.0;
    const double chi = a * a * rab;
    const double poa = p * b * rab;
    const double SKs = star ? SK : 0.0;
    // U*_k = chi U_k for the advected components, so F_k = U_k un + SK (chi - 1) U_k = U_k u_face with the
    // HLLC-consistent face velocity u_face = un + SK (chi - 1) (R8)
    const double uf = fma(SKs, chi - 1.0, un);
    const double U0 = z1 * r1, U1 = (1.0 - z1) * r2;
    F[0] = U0 * uf;
    F[1] = U1 * uf;
    F[2] = fma(rho * un, un, p) + SKs * rho * fma(chi, Sstar, -un);
    F[3] = rho * ut * uf;
    F[4] = fma(rhoE + p, un, SKs * fma(chi, fma(Sstar - un, fma(rho, Sstar, poa), rhoE), -rhoE));
    F[5] = z1 * uf;
    F[6] = U1 * lam * uf;
    F[7] = uf;
}

// state check of a finished cell on the high words (integer pipe): q0, q1 positive normal numbers, q2, q3, q4, q6 and the
// wavespeed finite.  (q5 was clamped just before and cannot be non-finite here.)
__device__ __forceinline__ bool state_ok(const double o[7], double a)
{
    const int pos = min(__double2hiint(o[0]), __double2hiint(o[1]));
    int m = max(__double2hiint(o[0]), __double2hiint(o[1]));
    m = max(m, max(__double2hiint(o[2]) & 0x7fffffff, __double2hiint(o[3]) & 0x7fffffff));
    m = max(m, max(__double2hiint(o[4]) & 0x7fffffff, __double2hiint(o[6]) & 0x7fffffff));
    m = max(m, __double2hiint(a) & 0x7fffffff);
    return pos > 0 && m < 0x7ff00000;
}

// finished cell of the second pass: trailing S(dt/2) (SRC != SRC_NONE), wavespeed of the new state, state check (a6, a7, R17)
template <int SRC, bool EX>
__device__ __forceinline__ void trail_cell(const Params& P, const double* __restrict__ tab, double o[7], double tau, double Tsafe, double& smax,
                                           int& bad, bool& hot)
{
    FCell W; double dE, q6n;
    prim_cell<SRC, EX>(P, tab, o, tau, Tsafe, W, dE, q6n, hot);
    o[4] += dE; o[6] = q6n;
    const double a = dmax_(fabs(W.un), fabs(W.ut)) + q_sqrt(W.rc2 * W.irho);
    bad |= state_ok(o, a) ? 0 : 1;
    smax = dmax_(smax, a);
}

// dt and tsafe of the running step.  They live in the control block that the LAST block of this very kernel rewrites for the
// next step (step_end_by_last_block) -- after every block has read them, the ticket sees to that -- so for the kernel as a whole
// the two words are neither read-only nor unaliased: no __restrict__ / LDG.NC on them and no load the compiler may repeat later,
// but exactly one L2 load per call of a segment function (the redo call reads the same, still unchanged, values again).
__device__ __forceinline__ double ld_ctl(const double* p)
{
    double v;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void reduce_smax(double smax, int bad, Ctl* ctl)
{
    for (int o = 16; o > 0; o >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(&ctl->smax_bits, dbits(smax));
        if (bad) atomicOr(&ctl->bad, 1);
    }
}

// post-source conserved values of a cell whose post-source lambda is known (pass 1 applies S on load, O6)
// O5 moves q1 Q (lam0 - lam1) with lam0 = clamp(q6/q1, 0, 1) (O3): q1 lam0 = q6 clamped to [0, q1]
__device__ __forceinline__ void lead_fix(const Params& P, double q[7], double lam1)
{
    const double q6n = q[1] * lam1;
    const double q6c = hi_word(q[6]) < 0 ? 0.0 : dmin_(q[6], q[1]);
    q[4] = fma(P.Q, q6c - q6n, q[4]);
    q[6] = q6n;
}

// ---------------------------------------------------------------------------------------------------------------
// end of a step: t, step counter, next dt from the max wavespeed (a7, R11) and the temperature bound below which the R13
// rule certainly gives n_sub = 1 for tau = dt/2.  Run by one thread: of k_ctl, or of the last block of the step's pass-2
// sweep to finish (step_end_by_last_block), which saves the launch.
// ---------------------------------------------------------------------------------------------------------------
__host__ __device__ inline double tsafe_for(double tau, double Cpre, double Ta, double theta0)
{
    // n_sub = 1 + floor(tau C g(Ta/T) / theta0), g(y) = 1/(1 + y + y^2/2 + y^3/6) decreasing in y.
    // Return T* such that T < T* guarantees tau C g < theta0 (1 - 1e-6); +inf when that holds for every T.
    const double target = theta0 * (1.0 - 1e-6) / (tau * Cpre);       // need g(y) < target
    if (!(tau > 0.0) || target >= 1.0) return 1e300;
    // y* = positive root of h(y) = 1 + y + y^2/2 + y^3/6 - 1/target (h' > 0, h'' > 0 for y > 0).  Newton from
    // y0 = cbrt(6/target), where h(y0) = 1 + y0 + y0^2/2 > 0: the iterates fall monotonically onto the root from the right,
    // so every one of them is a safe bound (y_n >= y*  =>  Ta/y_n <= Ta/y*).  A dozen divisions instead of the 64
    // bisections of round 1.
    const double r = 1.0 / target;
    double y = cbrt(6.0 * r);
    for (int it = 0; it < 12; ++it) {
        const double h = 1.0 + y * (1.0 + y * (0.5 + y * (1.0 / 6.0))) - r;
        const double dh = 1.0 + y * (1.0 + 0.5 * y);
        const double yn = y - h / dh;
        if (!(yn < y)) break;                                         // converged (or rounding would step back over the root)
        y = yn;
    }
    return Ta / (y * (1.0 + 1e-12));                                  // T < Ta/y  =>  Ta/T > y >= y*  =>  g < target
}

__device__ __forceinline__ void ctl_update(const Params& P, Ctl* ctl, int advance)
{
    if (advance) { ctl->t += ctl->dt; ctl->dt_last = ctl->dt; ctl->step += 1; }
    const double smax = __longlong_as_double((long long)atomicMax(&ctl->smax_bits, 0ull));    // (read at the point of coherence)
    const double dt = ctl->dt_fixed > 0.0 ? ctl->dt_fixed : P.cfl * P.hmin / smax;
    ctl->dt = dt;
    ctl->tsafe = P.reactive ? tsafe_for(0.5 * dt, P.Cpre, P.Ta, P.theta0) : 1e300;
    ctl->smax_bits = 0ull;
}

__global__ void k_ctl(const __grid_constant__ Params P, Ctl* ctl, int advance)
{
    pdl_launch_dependents();
    pdl_wait();
    ctl_update(P, ctl, advance);
}

// Last instruction block of a pass-2 sweep kernel: every block takes a ticket once its warps have added their wavespeed
// maxima; the block that takes the last one has seen all of them (fence, then ticket) and ends the step.  Every block has
// read dt long before (at its start), so overwriting ctl->dt here is safe; the next kernel starts after this one has ended.
__device__ __forceinline__ void step_end_by_last_block(const Params& P, Ctl* ctl)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned total = gridDim.x * gridDim.y;
        if (atomicAdd(&ctl->ticket, 1u) == total - 1u) {
            __threadfence();
            ctl_update(P, ctl, 1);
            ctl->ticket = 0u;
        }
    }
}

#ifndef NMSDT_Y_MINBLOCKS
#define NMSDT_Y_MINBLOCKS 2
#endif
#ifndef NMSDT_X_MINBLOCKS
#define NMSDT_X_MINBLOCKS 3
#endif
constexpr int XW = 4;                       // warps per block in k_xsweep
constexpr int RING = 33;
constexpr int XRAMP = 4;                    // cells left of a segment that k_xsweep recomputes (stencil radius 2, two passes of neighbours)
constexpr int RING_DOUBLES = (16 + 12 + 8) * RING;
constexpr int PRING = 66;                   // staged input pairs: chunk k (32 slots), chunk k+1 in flight, lane 31 of chunk k-1
constexpr int XS_DOUBLES = XW * (RING_DOUBLES + 7 * PRING * 2);    // dynamic part (the math tables are static)

} // namespace

// ---------------------------------------------------------------------------------------------------------------
// Boundary rules folded into the sweeps (a2; P:129 transmissive inflow, P:135 periodic top / bottom; R12): a ghost cell is
// never read from memory, its value is taken from the cell the rule names when the sweep loads it -- in the copies of the
// loop bodies that handle segment edges only, so the marching loops proper do not pay for it, and a step needs no halo
// launch.  Cell index c of a line of n cells, c in [-2, -1] or [n, n+1]:
//   transmissive (0): nearest interior cell;  periodic (1): c -+ n;  reflective (2): mirror image, normal momentum negated;
//   fixed inflow (3, x-lo only): the column captured by sim_init;  external (4, x only): the stored ghost column (a
//   neighbour slab's cells, written by the slab exchange).
// ghost_src returns the interior index the value comes from (and whether the normal momentum changes sign), or -1 when the
// stored / staged value is to be used as it is (interior cell, external side, fixed inflow -- handled by the caller).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int ghost_src(int c, int n, int bc_lo, int bc_hi, bool& flip)
{
    flip = false;
    if (c < 0) {
        if (bc_lo == 1) return ((c % n) + n) % n;
        if (bc_lo == 2) { flip = true; return min(-1 - c, n - 1); }
        return bc_lo == 0 ? 0 : -1;
    }
    if (c >= n) {
        if (bc_hi == 1) return (c - n) % n;
        if (bc_hi == 2) { flip = true; return max(2 * n - 1 - c, 0); }
        return bc_hi == 0 ? n - 1 : -1;
    }
    return -1;
}

// ---------------------------------------------------------------------------------------------------------------
// input staging: cp.async (x-sweep), bulk tensor copies + mbarriers (y-sweep)
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16(double* smem, const double* gmem)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// p + bytes as ONE 64-bit add the compiler may not take apart.  Left to itself it rebuilds every plane's address from a 64-bit
// element index (add, add-with-carry, shift-and-add, twice) -- 4-5 instructions per address, 7 addresses per load and per
// store; a chain of these costs 2 per address.
template <typename T>
__device__ __forceinline__ T* ptr_add(T* p, unsigned long long bytes)
{
    unsigned long long r;
    asm("add.u64 %0, %1, %2;" : "=l"(r) : "l"((unsigned long long)p), "l"(bytes));
    return (T*)r;
}

// TMA (cp.async.bulk.tensor) + mbarrier primitives of the y-sweep's input staging: one lane per warp arms the stage's
// barrier with the byte count and issues one bulk tensor copy per row -- a {32 columns, 1 row, 7 planes} box of the
// plane set (described by a CUtensorMap built in sim_create) -- instead of 7 cp.async + their 64-bit address
// arithmetic in every thread.
// (The helpers take 32-bit shared-space addresses: converting a generic pointer at every use costs ~18 instructions per row.)
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, int parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned smem_dst, const CUtensorMap* tm, int c0, int c1, int c2, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

// ---------------------------------------------------------------------------------------------------------------
// y-sweep (a5): thread per column, register marching
// ---------------------------------------------------------------------------------------------------------------
constexpr int YT = 256;      // threads (columns) per block in k_ysweep: 2 blocks of 8 warps per SM (one table copy per block)
constexpr int YST = 3;       // staged rows per thread: c-1 (re-read when its update starts), c, and c+1 in flight
constexpr int YS_DOUBLES = (YST * 7 + 16 + 11) * YT + 16;       // dynamic part (+ 128 bytes of alignment slack; the math tables and the barriers are static)

struct YPipe { int st, ph; };

// Per-thread state that lives across rows is kept in thread-private shared-memory slots ([..][YT] layout of value pairs,
// no barriers): the staged input rows, the primitive window (cell c-1 and its backward differences) and the previous
// right-face state.
// Only the half-finished update of cell c-1 stays in registers; this keeps the kernel at 128 registers (16 warps/SM).
// One column segment of the y-sweep (rows c0 .. c0+seg-1 of column col); returns whether a cell asked for RK4
// sub-stepping or the first-order fallback (EXACT = false only; the caller then redoes the segment with EXACT = true --
// the pass is out of place).
template <int MODE, bool EXACT, int LIM>
__device__ __forceinline__ bool y_segment(const Params& P, double* __restrict__ qout, const double* dtp, int seg, int col, const double* __restrict__ s_tab, double* __restrict__ s_dyn, double& smax, int& bad,
                                          const CUtensorMap* tm, unsigned bars, unsigned wmask, YPipe& pp)
{
    // staged input rows: per warp YST stages of [7 planes][32 columns], each filled by one bulk tensor copy;
    // thread-private slots, paired so that one 128-bit access moves two values: the window (W(c-1), 1/rho, rho c^2 and
    // the 7 differences W(c-1) - W(c-2): 8 pairs), the previous right-face state (5 pairs + c)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double (*s_st)[7][32] = reinterpret_cast<double (*)[7][32]>(s_dyn + warp * (YST * 7 * 32));
    double2 (*s_w2)[YT] = reinterpret_cast<double2 (*)[YT]>(s_dyn + YST * 7 * YT);
    double2 (*s_r2)[YT] = reinterpret_cast<double2 (*)[YT]>(s_dyn + (YST * 7 + 16) * YT);
    double* s_rc = s_dyn + (YST * 7 + 16 + 10) * YT;
    constexpr int SRC = (MODE == MODE_LEAD || MODE == MODE_TRAIL) ? (EXACT ? SRC_EXACT : SRC_FAST) : SRC_NONE;
    const int tid = threadIdx.x;
    bool hot = false;               // a cell needs the exact rules (R13 sub-steps or the R17 fallback): redo the segment
    const int c0 = blockIdx.y * seg, c1 = min(c0 + seg, P.ny);
    const double dt = ld_ctl(dtp), tau = 0.5 * dt, Tsafe = ld_ctl(dtp + 1);
    const double dtdx = dt / P.dy, khalf = 0.5 * dtdx;
    // (the plane stride as a 32-bit number -- sim_create refuses planes of 2^32 doubles -- so that a plane's address is ONE
    // IMAD.WIDE.U32 from the row pointer instead of a 64 x 64-bit product)
    const unsigned long long fs = (unsigned)P.fstride, fsb = fs * sizeof(double);
    const long long pitch = P.pitch;
    const unsigned long long pitchb = (unsigned long long)pitch * sizeof(double);
    double* pout = qout + (long long)(c0 + NGY) * pitch + NGX + col;
    const int nrows = c1 - c0 + 4;
    // one lane per warp stages a row: the {32, 1, 7} box at (first column of the warp, row, plane 0) of the input plane set.
    // `r` is the row of the grid, -2 .. ny + 1; a ghost row (only ever staged and read by the EDGE copy of the body) is taken
    // from the interior row the boundary rule names (ghost_src), its normal momentum negated on read where the wall reflects.
    const int tx = NGX + col - lane;
    const unsigned st_addr = smem_u32(&s_st[0][0][0]);    // shared-space addresses of the warp's stages (1792 B each) and barriers
    auto stage_row = [&](int sg, int r, bool edge) {
        if (lane == 0) {
            bool flip;
            const int src = edge ? ghost_src(r, P.ny, P.bc_ylo, P.bc_yhi, flip) : -1;
            mbar_expect_tx(bars + 8u * sg, 7 * 32 * (int)sizeof(double));
            tma_load_3d(st_addr + (unsigned)(7 * 32 * sizeof(double)) * sg, tm, tx, (src >= 0 ? src : r) + NGY, 0, bars + 8u * sg);
        }
    };
    auto read_row = [&](int sg, double q[7]) {            // sweep field order: q0, q1, q3 (normal), q2 (tangential), q4, q5, q6
        q[0] = s_st[sg][0][lane]; q[1] = s_st[sg][1][lane]; q[2] = s_st[sg][3][lane]; q[3] = s_st[sg][2][lane];
        q[4] = s_st[sg][4][lane]; q[5] = s_st[sg][5][lane]; q[6] = s_st[sg][6][lane];
    };
    auto reflected = [&](int r) { return (r < 0 && P.bc_ylo == 2) || (r >= P.ny && P.bc_yhi == 2); };
    int st = pp.st, ph = pp.ph;                   // stage of row jj and the parity of its barrier's current phase
    stage_row(st, c0 - 2, true);
    double acc[7] = {0, 0, 0, 0, 0, 0, 0}, z1n = 0.0;
    auto row = [&](auto edge_tag, int jj) {       // row c = c0 - 2 + jj; EDGE: a ramp-up row or one of the last 3 (see below)
        constexpr bool EDGE = decltype(edge_tag)::value;
        const int sn = st == YST - 1 ? 0 : st + 1, sp = st == 0 ? YST - 1 : st - 1;
        if (!EDGE || jj + 1 < nrows) {
            __syncwarp(wmask);                    // every lane is done with stage sn (row jj - 2, last read in the previous iteration)
            stage_row(sn, c0 - 1 + jj, EDGE);
        }
        mbar_wait(bars + 8u * st, ph);
        FCell Wp;
        {
            double q[7];
            read_row(st, q);
            if (EDGE && reflected(c0 - 2 + jj)) q[2] = -q[2];
            double dE, q6n;
            prim_cell<MODE == MODE_LEAD ? SRC : SRC_NONE, EXACT>(P, s_tab, q, tau, Tsafe, Wp, dE, q6n, hot);
        }
        double WL[7], WR[7], lam0c;
        {                                         // centre cell c-1: s_w[0] = W(c-1), s_w[1][0..6] = W(c-1) - W(c-2)
            FCell W0;
            double a[7];
            {
                const double2 w0 = s_w2[0][tid], w1 = s_w2[1][tid], w2 = s_w2[2][tid], w3 = s_w2[3][tid];
                const double2 w4 = s_w2[4][tid], w5 = s_w2[5][tid], w6 = s_w2[6][tid], w7 = s_w2[7][tid];
                W0.r1 = w0.x; W0.r2 = w0.y; W0.un = w1.x; W0.ut = w1.y; W0.p = w2.x; W0.z1 = w2.y; W0.lam = w3.x; W0.irho = w3.y;
                W0.rc2 = w4.x; a[0] = w4.y; a[1] = w5.x; a[2] = w5.y; a[3] = w6.x; a[4] = w6.y; a[5] = w7.x; a[6] = w7.y;
            }
            const double b[7] = {Wp.r1 - W0.r1, Wp.r2 - W0.r2, Wp.un - W0.un, Wp.ut - W0.ut, Wp.p - W0.p, Wp.z1 - W0.z1, Wp.lam - W0.lam};
            lam0c = W0.lam;
            recon_core<LIM, EXACT>(P, W0, a, b, khalf, WL, WR, !EDGE || jj >= 2, hot);      // rows 0, 1: the window is not real yet
            s_w2[0][tid] = make_double2(Wp.r1, Wp.r2); s_w2[1][tid] = make_double2(Wp.un, Wp.ut); s_w2[2][tid] = make_double2(Wp.p, Wp.z1);
            s_w2[3][tid] = make_double2(Wp.lam, Wp.irho); s_w2[4][tid] = make_double2(Wp.rc2, b[0]); s_w2[5][tid] = make_double2(b[1], b[2]);
            s_w2[6][tid] = make_double2(b[3], b[4]); s_w2[7][tid] = make_double2(b[5], b[6]);
        }
        FFace fl, fr, pr;
        bool oor = false;                         // a face density outside the power tables (only counted once the window is real)
        face_fast<EXACT, true>(P, s_tab, WL, fl, oor);
        face_fast<EXACT, true>(P, s_tab, WR, fr, oor);
        hot |= oor && (!EDGE || jj >= 2);
        {
            const double2 r0 = s_r2[0][tid], r1 = s_r2[1][tid], r2 = s_r2[2][tid], r3 = s_r2[3][tid], r4 = s_r2[4][tid];
            pr.r1 = r0.x; pr.r2 = r0.y; pr.un = r1.x; pr.ut = r1.y; pr.p = r2.x; pr.z1 = r2.y; pr.lam = r3.x; pr.rho = r3.y;
            pr.xC = r4.x; pr.xD = r4.y; pr.c = s_rc[tid];
        }
        s_r2[0][tid] = make_double2(fr.r1, fr.r2); s_r2[1][tid] = make_double2(fr.un, fr.ut); s_r2[2][tid] = make_double2(fr.p, fr.z1);
        s_r2[3][tid] = make_double2(fr.lam, fr.rho); s_r2[4][tid] = make_double2(fr.xC, fr.xD); s_rc[tid] = fr.c;
        double F[8];
        hllc_fast<true>(P, pr, fl, F);                     // face between cells c-2 and c-1
        {                                         // finish cell c-2
            double o[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) o[k] = fma(-dtdx, F[k], acc[k]);
            o[5] = fma(dtdx * z1n, F[7], o[5]);                           // R8: non-conservative z1 term
            o[5] = clampf(o[5], P.z_min, P.z_max);
            const bool valid = !EDGE || jj >= 4;             // (the ramp-up rows finish nothing)
            if (MODE == MODE_TRAIL || MODE == MODE_TRAIL_INERT) {
                double sm1 = 0.0; int bad1 = 0; bool hot1 = false;
                trail_cell<MODE == MODE_TRAIL ? SRC : SRC_NONE, EXACT>(P, s_tab, o, tau, Tsafe, sm1, bad1, hot1);
                smax = valid ? dmax_(smax, sm1) : smax;
                bad |= valid ? bad1 : 0;
                hot |= valid && hot1;
            }
            if (valid) {
                double* po = pout;                // planes 0 .. 6 hold q0, q1, q2 (tangential here), q3 (normal), q4, q5, q6
                *po = o[0]; po = ptr_add(po, fsb); *po = o[1]; po = ptr_add(po, fsb); *po = o[3]; po = ptr_add(po, fsb); *po = o[2];
                po = ptr_add(po, fsb); *po = o[4]; po = ptr_add(po, fsb); *po = o[5]; po = ptr_add(po, fsb); *po = o[6];
                pout = ptr_add(pout, pitchb);
            }
        }
        {                                         // start cell c-1 with its lower-face flux
            double o[7];
            read_row(sp, o);                      // (row jj - 1 is a cell of the segment whenever what starts here is kept: no ghost rule)
            if (MODE == MODE_LEAD) lead_fix(P, o, lam0c);
            z1n = o[5];
#pragma unroll
            for (int k = 0; k < 7; ++k) acc[k] = fma(dtdx, F[k], o[k]);
            acc[5] = fma(-dtdx * z1n, F[7], acc[5]);
        }
        st = sn;
        ph ^= sn == 0 ? 1 : 0;
    };
    // EDGE copy of the body: the 4 ramp-up rows, which run on a window / face / flux that is not real yet (finite or
    // not: nothing is stored or counted), and the last 3 rows, which stage and read the rows beyond the segment end -- ghost rows
    // when the segment ends at the grid's.  The rows in between touch cells of the grid only.
    // (one call site per copy: a second one makes the compiler call the body instead of inlining it, and everything it captures
    // -- the running update, the pipeline state -- then lives in local memory)
    for (int jj = 0; jj < nrows; ++jj) {
        if (jj < 4 || jj >= nrows - 3) row(std::true_type{}, jj);
        else row(std::false_type{}, jj);
    }
    pp.st = st; pp.ph = ph;                       // (a redo of the segment goes on from here: every staged row has been consumed)
    return hot;
}

template <int MODE, int LIM>
__global__ void __launch_bounds__(YT, NMSDT_Y_MINBLOCKS) k_ysweep(const __grid_constant__ Params P, const __grid_constant__ CUtensorMap tm,
                                                                  double* __restrict__ qout, const double* dtp, Ctl* ctl, int seg, int end_step)
{
    extern __shared__ __align__(16) double s_dyn_raw[];
    // the staged rows are bulk-copy destinations and must be 128-byte aligned: the dynamic part follows the static arrays
    // below at whatever offset their sizes leave, so it carries 128 spare bytes and starts at the next multiple of 128
    double* s_dyn = s_dyn_raw + ((128u - (smem_u32(s_dyn_raw) & 127u)) & 127u) / sizeof(double);
    __shared__ __align__(16) double s_tab[MATH_TAB_DOUBLES];     // static: table lookups address it as [idx + const]
    __shared__ __align__(8) unsigned long long s_bar[YT / 32][YST];
    pdl_launch_dependents();
    for (int i = threadIdx.x; i < MATH_TAB_DOUBLES; i += blockDim.x) s_tab[i] = P.tab[i];
    if (threadIdx.x < (YT / 32) * YST) mbar_init(smem_u32(&s_bar[0][0] + threadIdx.x), 1);
    fence_proxy_async();
    __syncthreads();
    pdl_wait();                                                  // the state, dt and the control block belong to the previous kernel until here
    const int col = blockIdx.x * YT + threadIdx.x;
    const unsigned wmask = __ballot_sync(0xffffffffu, col < P.nx);
    double smax = 0.0; int bad = 0;
    if (col < P.nx) {
        YPipe pp{0, 0};
        const unsigned bars = smem_u32(s_bar[threadIdx.x >> 5]);
        const bool redo = y_segment<MODE, false, LIM>(P, qout, dtp, seg, col, s_tab, s_dyn, smax, bad, &tm, bars, wmask, pp);
        if (__any_sync(wmask, redo)) {                           // rare: redo the warp's segment with the exact R13 / R17 rules
            if ((threadIdx.x & 31) == 0) atomicAdd(&ctl->redo, 1);
            smax = 0.0; bad = 0;
            y_segment<MODE, true, LIM>(P, qout, dtp, seg, col, s_tab, s_dyn, smax, bad, &tm, bars, wmask, pp);
        }
    }
    if (MODE == MODE_TRAIL || MODE == MODE_TRAIL_INERT) {
        reduce_smax(smax, bad, ctl);
        if (end_step) step_end_by_last_block(P, ctl);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// x-sweep (a4): warp per row segment, 2 cells per lane, shared-memory rings between lanes
// ---------------------------------------------------------------------------------------------------------------
// One row segment of the x-sweep (cells c0 .. c0+seg-1 of row `row`, one warp); returns whether a cell asked for RK4
// sub-stepping or the first-order fallback (EXACT = false only; the caller then redoes the segment with EXACT = true --
// the pass is out of place).
template <int MODE, bool EXACT, int LIM>
__device__ __forceinline__ bool x_segment(const Params& P, const double* __restrict__ qin, double* __restrict__ qout, const double* dtp,
                                          int seg, int row, const double* __restrict__ s_tab, double* __restrict__ s_dyn, double& smax, int& bad)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int SRC = (MODE == MODE_LEAD || MODE == MODE_TRAIL) ? (EXACT ? SRC_EXACT : SRC_FAST) : SRC_NONE;
    constexpr bool XDEFER = MODE != MODE_TRAIL;         // (see FFace)
    double* s_ring = s_dyn;
    bool hot = false;               // a cell needs the exact rules (R13 sub-steps or the R17 fallback): redo the segment
    // rings of value PAIRS (one 128-bit access moves two values)
    double2* rw = reinterpret_cast<double2*>(s_ring + warp * RING_DOUBLES);   // [8][33]: W of the lane's cells A (0-6), B (7-13), 1/rho_B, (rho c^2)_B
    double2* rfr = rw + 8 * RING;                    // [6][33]: right-face state of cell A (11 values)
    double2* rf = rfr + 6 * RING;                    // [4][33]: flux of face A-1/2
    double2* stg = reinterpret_cast<double2*>(s_dyn + XW * RING_DOUBLES) + warp * 7 * PRING;   // [7][66] input pairs
    const int c0 = blockIdx.y * seg, c1 = min(c0 + seg, P.nx);
    const double dt = ld_ctl(dtp), tau = 0.5 * dt, Tsafe = ld_ctl(dtp + 1);
    const double dtdx = dt / P.dx, khalf = 0.5 * dtdx;
    const unsigned long long fs = (unsigned)P.fstride;     // (32-bit plane stride: see y_segment)
    const unsigned long long fsb = fs * sizeof(double);
    const double* rin = qin + (long long)(row + NGY) * P.pitch + NGX;
    double* rout = qout + (long long)(row + NGY) * P.pitch + NGX;
    const int nxe = (P.nx + 1) & ~1;                 // last pair base that is ever needed (cell nx+1 is the outer ghost; for odd nx the pair ends in row padding)
    const int niter = (c1 - c0 + XRAMP + 63) >> 6;   // chunks of 64 cells, the first one starts XRAMP = 4 cells left of c0
    const bool fixed_in = (MODE == MODE_LEAD) && (P.bc_xlo == 3);
    int sw = lane;                                   // ring slot written by this lane: (32 k + lane) mod 33
    int ps = lane;                                   // staging slot of this lane's pair: (32 k + lane) mod 66
    {   // stage chunk 0 (cells c0-2 .. c0+61)
        const int Ac = min(max(c0 - XRAMP + 2 * lane + 2, -2), nxe);
#pragma unroll
        for (int f = 0; f < 7; ++f) cp_async16(reinterpret_cast<double*>(stg + f * PRING + ps), rin + Ac + f * fs);
        cp_async_commit();
    }
    // EDGE: the first chunk of the segment (ramp-up: lanes 0, 1 update nothing; ghost cells of the row start) and the last one or
    // two (which end inside the chunk, at the row end, in the ghost cells: those get their values from the boundary rule).  Every chunk in between updates 64 cells of the segment from 68 cells that all
    // exist, so its copy of the body carries none of the validity predicates.
    auto chunk = [&](auto edge_tag, int k) {
        constexpr bool EDGE = decltype(edge_tag)::value;
        const int b = c0 - XRAMP + 64 * k;           // first cell this iteration would update
        const int A = b + 2 * lane + 2;              // this lane loads cells A, A+1 and reconstructs cells A-1, A
        // In iteration 0 lanes 0, 1 hold the left stencil cells c0-2 .. c0+1: they have no (complete) left neighbours of
        // their own, so what they would update (cells c0-4 .. c0-1, another segment's) is not stored; the body is branch
        // free and simply runs on not-yet-valid ring data there.  Like the y-sweep, a segment costs 4 ramp-up cells.
        const int sr = sw == 0 ? RING - 1 : sw - 1;  // left neighbour's slot
        FCell WA, WB;
        const int psn = ps + 32 >= PRING ? ps + 32 - PRING : ps + 32;
        if (k + 1 < niter) {                         // stage the next chunk while this one is computed
            const double* gp = rin + min(A + 64, nxe);      // one 64-bit pointer, then a chain of plane strides
#pragma unroll
            for (int f = 0; f < 7; ++f, gp = ptr_add(gp, fsb)) cp_async16(reinterpret_cast<double*>(stg + f * PRING + psn), gp);
        }
        cp_async_commit();
        cp_async_wait<1>();
        // ---- phase 1: primitives (+ leading source) of the staged pair -----------------------------------------
        {
            const int Ac = EDGE ? min(max(A, -2), nxe) : A;
            double qa[7], qb[7];
#pragma unroll
            for (int f = 0; f < 7; ++f) { const double2 v = stg[f * PRING + ps]; qa[f] = v.x; qb[f] = v.y; }
            if (EDGE && (Ac < 0 || Ac + 1 >= P.nx)) {              // a ghost cell in the pair: apply the boundary rule (see ghost_src)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int c = Ac + h;
                    double* q = h == 0 ? qa : qb;
                    if (c > P.nx + 1) continue;                   // row padding (odd nx): not a cell, never used
                    bool flip;
                    const int src = ghost_src(c, P.nx, P.bc_xlo, P.bc_xhi, flip);
                    if (src >= 0) {
#pragma unroll
                        for (int f = 0; f < 7; ++f) q[f] = rin[src + f * fs];
                        if (flip) q[2] = -q[2];
                    } else if (c < 0 && P.bc_xlo == 3) {
#pragma unroll
                        for (int f = 0; f < 7; ++f) q[f] = P.inflow[f * P.ny + row];
                    }
                }
            }
            double dE, q6n;
            bool hotb = false;                       // cell Ac + 1 = nx + 2 (odd nx) is row padding, not a cell
            prim_cell<MODE == MODE_LEAD ? SRC : SRC_NONE, EXACT>(P, s_tab, qa, (EDGE && fixed_in && Ac < 0) ? 0.0 : tau, Tsafe, WA, dE, q6n, hot);
            prim_cell<MODE == MODE_LEAD ? SRC : SRC_NONE, EXACT>(P, s_tab, qb, (EDGE && fixed_in && Ac + 1 < 0) ? 0.0 : tau, Tsafe, WB, dE, q6n, hotb);
            hot |= hotb && (!EDGE || Ac <= P.nx);
            rw[0 * RING + sw] = make_double2(WA.r1, WA.r2); rw[1 * RING + sw] = make_double2(WA.un, WA.ut);
            rw[2 * RING + sw] = make_double2(WA.p, WA.z1);  rw[3 * RING + sw] = make_double2(WA.lam, WB.r1);
            rw[4 * RING + sw] = make_double2(WB.r2, WB.un); rw[5 * RING + sw] = make_double2(WB.ut, WB.p);
            rw[6 * RING + sw] = make_double2(WB.z1, WB.lam); rw[7 * RING + sw] = make_double2(WB.irho, WB.rc2);
        }
        __syncwarp();
        // ---- phase 2: reconstruct cells A-1 and A, four face states ------------------------------------------
        FFace FL1, FR1, FL2;
        double lam_u0 = 0.0, lam_u1 = 0.0;
        {
            FCell Wmm, Wm1;
            {
                const double2 v0 = rw[0 * RING + sr], v1 = rw[1 * RING + sr], v2 = rw[2 * RING + sr], v3 = rw[3 * RING + sr];
                const double2 v4 = rw[4 * RING + sr], v5 = rw[5 * RING + sr], v6 = rw[6 * RING + sr], v7 = rw[7 * RING + sr];
                Wmm.r1 = v0.x; Wmm.r2 = v0.y; Wmm.un = v1.x; Wmm.ut = v1.y; Wmm.p = v2.x; Wmm.z1 = v2.y; Wmm.lam = v3.x;
                Wmm.irho = 0.0; Wmm.rc2 = 0.0;
                Wm1.r1 = v3.y; Wm1.r2 = v4.x; Wm1.un = v4.y; Wm1.ut = v5.x; Wm1.p = v5.y; Wm1.z1 = v6.x; Wm1.lam = v6.y;
                Wm1.irho = v7.x; Wm1.rc2 = v7.y;
            }
            lam_u0 = Wmm.lam; lam_u1 = Wm1.lam;
            double WL[7], WR[7];
            // What may ask for a redo: reconstructions whose window is real (k = 0, lane 0: the left slot is not written yet)
            // and whose cell is at most the ghost cell nx, the last one a stored face needs.  Cell nx + 1 is reconstructed
            // from cell nx + 2, which does not exist: row padding when nx is odd (its NaN primitives would raise the
            // out-of-table flag on every row end), a clamped reload otherwise.
            const bool real = !EDGE || k > 0 || lane > 0;
            const bool cnt1 = !EDGE || (real && A - 1 <= P.nx), cnt2 = !EDGE || (real && A <= P.nx);
            bool oor1 = false, oor2 = false;         // a face density outside the power tables
            recon_fast<LIM, EXACT>(P, Wmm, Wm1, WA, khalf, WL, WR, cnt1, hot);
            face_fast<EXACT, XDEFER>(P, s_tab, WL, FL1, oor1);
            face_fast<EXACT, XDEFER>(P, s_tab, WR, FR1, oor1);
            recon_fast<LIM, EXACT>(P, Wm1, WA, WB, khalf, WL, WR, cnt2, hot);
            face_fast<EXACT, XDEFER>(P, s_tab, WL, FL2, oor2);
            FFace FR2;
            face_fast<EXACT, XDEFER>(P, s_tab, WR, FR2, oor2);
            hot |= (oor1 && cnt1) || (oor2 && cnt2);
            rfr[0 * RING + sw] = make_double2(FR2.r1, FR2.r2); rfr[1 * RING + sw] = make_double2(FR2.un, FR2.ut);
            rfr[2 * RING + sw] = make_double2(FR2.p, FR2.z1);  rfr[3 * RING + sw] = make_double2(FR2.lam, FR2.rho);
            rfr[4 * RING + sw] = XDEFER ? make_double2(FR2.xC, FR2.xD) : make_double2(FR2.rhoE, 0.0); rfr[5 * RING + sw] = make_double2(FR2.c, 0.0);
        }
        __syncwarp();
        // ---- phase 3: faces A-3/2 and A-1/2 ---------------------------------------------------------------------
        double F1[8], F2[8];
        {
            FFace FRp;
            {
                const double2 v0 = rfr[0 * RING + sr], v1 = rfr[1 * RING + sr], v2 = rfr[2 * RING + sr], v3 = rfr[3 * RING + sr];
                const double2 v4 = rfr[4 * RING + sr], v5 = rfr[5 * RING + sr];
                FRp.r1 = v0.x; FRp.r2 = v0.y; FRp.un = v1.x; FRp.ut = v1.y; FRp.p = v2.x; FRp.z1 = v2.y; FRp.lam = v3.x; FRp.rho = v3.y;
                FRp.xC = v4.x; FRp.xD = v4.y; FRp.rhoE = v4.x; FRp.c = v5.x;
            }
            hllc_fast<XDEFER>(P, FRp, FL1, F1);
            hllc_fast<XDEFER>(P, FR1, FL2, F2);
#pragma unroll
            for (int f = 0; f < 4; ++f) rf[f * RING + sw] = make_double2(F2[2 * f], F2[2 * f + 1]);
        }
        __syncwarp();
        // ---- phase 4: update cells A-2 = b + 2 lane and A-1 ---------------------------------------------------
        const int u0 = b + 2 * lane;
        {
            const bool valid = !EDGE || (u0 >= c0 && u0 < c1);
            double F0[8];
#pragma unroll
            for (int f = 0; f < 4; ++f) { const double2 v = rf[f * RING + sr]; F0[2 * f] = v.x; F0[2 * f + 1] = v.y; }
            const int pl = ps == 0 ? PRING - 1 : ps - 1;      // the pair staged by the left neighbour = cells u0, u0+1
            double oa[7], ob[7];
#pragma unroll
            for (int f = 0; f < 7; ++f) { const double2 v = stg[f * PRING + pl]; oa[f] = v.x; ob[f] = v.y; }
            if (MODE == MODE_LEAD) {
                lead_fix(P, oa, lam_u0);
                lead_fix(P, ob, lam_u1);
            }
            const double za = oa[5], zb = ob[5];
#pragma unroll
            for (int f = 0; f < 7; ++f) { oa[f] = fma(-dtdx, F1[f] - F0[f], oa[f]); ob[f] = fma(-dtdx, F2[f] - F1[f], ob[f]); }
            oa[5] = clampf(fma(dtdx * za, F1[7] - F0[7], oa[5]), P.z_min, P.z_max);       // R8
            ob[5] = clampf(fma(dtdx * zb, F2[7] - F1[7], ob[5]), P.z_min, P.z_max);
            const bool two = !EDGE || u0 + 1 < c1;
            if (MODE == MODE_TRAIL || MODE == MODE_TRAIL_INERT) {
                double sm1 = 0.0, sm2 = 0.0; int bad1 = 0, bad2 = 0; bool hot1 = false, hot2 = false;
                trail_cell<MODE == MODE_TRAIL ? SRC : SRC_NONE, EXACT>(P, s_tab, oa, tau, Tsafe, sm1, bad1, hot1);
                trail_cell<MODE == MODE_TRAIL ? SRC : SRC_NONE, EXACT>(P, s_tab, ob, tau, Tsafe, sm2, bad2, hot2);
                sm1 = valid ? sm1 : 0.0; sm2 = (valid && two) ? sm2 : 0.0;
                smax = dmax_(smax, dmax_(sm1, sm2));
                bad |= (valid ? bad1 : 0) | ((valid && two) ? bad2 : 0);
                hot |= (valid && hot1) || (valid && two && hot2);
            }
            // always a 128-bit pair store: only the last pair of a row with odd nx has a second cell that is not a cell, and that
            // one is the ghost column nx of the output planes, which the halo step (or the slab exchange) rewrites before any
            // x-sweep reads it and which nothing else reads
            double* po = rout + u0;
            if (valid) {
#pragma unroll
                for (int f = 0; f < 7; ++f, po = ptr_add(po, fsb)) *reinterpret_cast<double2*>(po) = make_double2(oa[f], ob[f]);
            }
        }
        sw = sw == 0 ? RING - 1 : sw - 1;            // (32 (k+1) + lane) mod 33
        ps = psn;
    };
    for (int k = 0; k < niter; ++k) {
        // a middle chunk loads cells b + 2 .. b + 65, all of them cells of the row below the segment end
        if (k == 0 || c0 - XRAMP + 64 * k + 65 >= c1) chunk(std::true_type{}, k);
        else chunk(std::false_type{}, k);
    }
    cp_async_wait<0>();
    return hot;
}

template <int MODE, int LIM>
__global__ void __launch_bounds__(32 * XW, NMSDT_X_MINBLOCKS) k_xsweep(const __grid_constant__ Params P, const double* __restrict__ qin, double* __restrict__ qout,
                                                    const double* dtp, Ctl* ctl, int seg, int end_step)
{
    extern __shared__ __align__(16) double s_dyn[];
    __shared__ __align__(16) double s_tab[MATH_TAB_DOUBLES];
    pdl_launch_dependents();
    for (int i = threadIdx.x; i < MATH_TAB_DOUBLES; i += blockDim.x) s_tab[i] = P.tab[i];
    __syncthreads();
    pdl_wait();
    const int row = blockIdx.x * XW + (threadIdx.x >> 5);
    double smax = 0.0; int bad = 0;
    if (row < P.ny) {
        const bool redo = x_segment<MODE, false, LIM>(P, qin, qout, dtp, seg, row, s_tab, s_dyn, smax, bad);
        if (__any_sync(0xffffffffu, redo)) {                     // rare: redo the warp's segment with the exact R13 / R17 rules
            if ((threadIdx.x & 31) == 0) atomicAdd(&ctl->redo, 1);
            smax = 0.0; bad = 0;
            __syncwarp();
            x_segment<MODE, true, LIM>(P, qin, qout, dtp, seg, row, s_tab, s_dyn, smax, bad);
        }
    }
    if (MODE == MODE_TRAIL || MODE == MODE_TRAIL_INERT) {
        reduce_smax(smax, bad, ctl);
        if (end_step) step_end_by_last_block(P, ctl);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// pointwise source step with the fused-path arithmetic (sim_source under SIM_VARIANT_FUSED), in place
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_source_fast(const __grid_constant__ Params P, double* __restrict__ q, const double* __restrict__ dtp)
{
    __shared__ double s_tab[MATH_TAB_DOUBLES];
    for (int i = threadIdx.x; i < MATH_TAB_DOUBLES; i += blockDim.x) s_tab[i] = P.tab[i];
    __syncthreads();
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (i >= P.nx) return;
    const long long id = (long long)(j + NGY) * P.pitch + NGX + i;
    double c[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) c[k] = q[k * P.fstride + id];
    FCell W; double dE, q6n; bool hot = false;
    prim_cell<SRC_EXACT>(P, s_tab, c, dtp[0], dtp[1], W, dE, q6n, hot);
    q[4 * P.fstride + id] = c[4] + dE;
    q[6 * P.fstride + id] = q6n;
}

// ---------------------------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------------------------
// Segment length along the marching axis.  A block marches over `seg` cells after `ramp` cells of ramp-up (recomputed
// halo) and a start that costs about `start` iterations (table copy, first staged row); `lines` blocks stand side by side,
// and up to `maxb` blocks are resident per SM.  With B = lines * nseg blocks:
//   * B > nsm * maxb (large grids): ceil(B / (nsm maxb)) waves of (seg + ramp + start) iterations, each at the throughput-bound
//     pace of maxb resident blocks -- large grids end up near `target`, with little ramp-up redundancy;
//   * otherwise one wave with b = ceil(B / nsm) blocks per SM, whose iterations take max(lat, b) / maxb of that pace: a lone
//     block is bound by the latency of the cell's dependency chain (measured in round 1 with 4 resident blocks per SM in both
//     directions: an iteration of a lone block took 2.6 (y, 128 columns) and 2.5 (x) times as long as its share of a full SM's.
//     The unit of `lat` is one block's share, 1/maxb of the SM: the y-sweep now runs 256-column blocks, 2 per SM -- a lone one
//     has twice the warps in flight and the same latency-bound iteration time, which is 2.6 x 2/4 = 1.3 of ITS share; that is
//     the 1.3 launch_sweep_fused passes, rescaled, not measured again), so small grids are cut into as many short segments as the SMs
//     can take before throughput binds -- on a machine that is not full, recomputed ramp-up cells are free and latency counts
//     (C1: 6 instead of 12 rows per block).
static double seg_cost(long long B, double iters, int nsm, int maxb, double lat)
{
    const long long b = (B + nsm - 1) / nsm;
    if (b <= maxb) return iters * (lat > (double)b ? lat : (double)b);
    return (double)((B + (long long)nsm * maxb - 1) / ((long long)nsm * maxb)) * iters * maxb;
}

static int pick_seg(int n, int target, int ramp, double start, int lines, int nsm, int maxb, double lat)
{
    int best_seg = n; double best = 1e300;
    for (int seg = n < 2 ? n : 2; seg <= n; ++seg) {
        if (seg > 2 * target) break;
        const int nseg = (n + seg - 1) / seg;
        const double cost = seg_cost((long long)lines * nseg, seg + ramp + start, nsm, maxb, lat);
        if (cost < best * (1.0 - 1e-9)) { best = cost; best_seg = seg; }
    }
    return best_seg;
}

// x-sweep: a segment of 64 m - XRAMP cells takes exactly m marching iterations of 64 cells (the first chunk starts XRAMP
// cells to the left) after a start (table copy, first staged chunk) that costs about two iterations.  Segment starts stay
// even (128-bit pair loads).
static int pick_seg_x(int n, int lines, int nsm, int maxb, double lat)
{
    const int mmax = (n + XRAMP + 63) / 64;                    // one segment for the whole row
    int best = 64 * mmax - XRAMP; double bestc = 1e300;
    for (int m = 1; m <= mmax; ++m) {
        const int seg = 64 * m - XRAMP;
        if (seg > 4096 && m < mmax) continue;                  // segments of at most a few thousand cells, or the whole row
        const int nseg = (n + seg - 1) / seg;
        const double cost = seg_cost((long long)lines * nseg, m + 2.0, nsm, maxb, lat);
        if (cost < bestc * (1.0 - 1e-9)) { bestc = cost; best = seg; }
    }
    return best;
}

static int num_sms()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0; cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    }
    return n;
}

template <int MODE, int LIM>
static void x_launch(bool attr_only, dim3 grid, size_t sm, cudaStream_t s, bool pdl, const Params& P, const double* qin, double* qout, const double* dtp,
                     Ctl* ctl, int seg, int end_step)
{
    if (attr_only) cudaFuncSetAttribute(k_xsweep<MODE, LIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    else launch_k(k_xsweep<MODE, LIM>, grid, dim3(32 * XW), sm, s, pdl, P, qin, qout, dtp, ctl, seg, end_step);
}
template <int MODE, int LIM>
static void y_launch(bool attr_only, dim3 grid, size_t sm, cudaStream_t s, bool pdl, const Params& P, const CUtensorMap* tm, double* qout, const double* dtp,
                     Ctl* ctl, int seg, int end_step)
{
    if (attr_only) cudaFuncSetAttribute(k_ysweep<MODE, LIM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    else launch_k(k_ysweep<MODE, LIM>, grid, dim3(YT), sm, s, pdl, P, *tm, qout, dtp, ctl, seg, end_step);
}

// dispatch on (direction, pass kind, limiter); attr_only = opt in to the dynamic shared memory instead of launching
static void sweep_dispatch(bool attr_only, int dir, int mode, int lim, dim3 grid, cudaStream_t s, bool pdl, const Params& P, const double* qin,
                           const CUtensorMap* tm, double* qout, const double* dtp, Ctl* ctl, int seg, int end_step)
{
    const size_t sm = (dir == 0 ? XS_DOUBLES : YS_DOUBLES) * sizeof(double);
#define NMSDT_CASE(D, M, L)                                                                                          \
    if (dir == D && mode == M && lim == L) {                                                                        \
        if (D == 0) x_launch<M, L>(attr_only, grid, sm, s, pdl, P, qin, qout, dtp, ctl, seg, end_step);                   \
        else        y_launch<M, L>(attr_only, grid, sm, s, pdl, P, tm, qout, dtp, ctl, seg, end_step);                   \
        return;                                                                                                     \
    }
    NMSDT_CASE(0, MODE_PLAIN, 0) NMSDT_CASE(0, MODE_LEAD, 0) NMSDT_CASE(0, MODE_TRAIL, 0) NMSDT_CASE(0, MODE_TRAIL_INERT, 0)
    NMSDT_CASE(0, MODE_PLAIN, 1) NMSDT_CASE(0, MODE_LEAD, 1) NMSDT_CASE(0, MODE_TRAIL, 1) NMSDT_CASE(0, MODE_TRAIL_INERT, 1)
    NMSDT_CASE(1, MODE_PLAIN, 0) NMSDT_CASE(1, MODE_LEAD, 0) NMSDT_CASE(1, MODE_TRAIL, 0) NMSDT_CASE(1, MODE_TRAIL_INERT, 0)
    NMSDT_CASE(1, MODE_PLAIN, 1) NMSDT_CASE(1, MODE_LEAD, 1) NMSDT_CASE(1, MODE_TRAIL, 1) NMSDT_CASE(1, MODE_TRAIL_INERT, 1)
#undef NMSDT_CASE
}

// opt in to the dynamic shared memory the sweeps need (called once per handle from sim_create, outside any capture)
void init_fused_kernels()
{
    Params P{};
    for (int dir = 0; dir < 2; ++dir)
        for (int mode = 0; mode < 4; ++mode)
            for (int lim = 0; lim < 2; ++lim) sweep_dispatch(true, dir, mode, lim, dim3(1), nullptr, false, P, nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0);
}

// mode 0 plain, 1 leading source on load, 2 trailing source + max-wavespeed partial.  An inert run (P.reactive = 0) has
// no source step: its pass 1 is the plain sweep and its pass 2 the sweep + wavespeed.  The limiter (R5) is a template
// parameter so that the marching loop stays one basic block.
void launch_sweep_fused(const Params& P, const double* qin, const CUtensorMap* tm_in, double* qout, const double* dtp, Ctl* ctl, int dir, int mode, cudaStream_t s,
                        bool pdl, bool end_step)
{
    if (!P.reactive) mode = mode == MODE_LEAD ? MODE_PLAIN : (mode == MODE_TRAIL ? MODE_TRAIL_INERT : mode);
    const int lim = P.limiter == 0 ? 0 : 1;
    if (dir == 0) {
        const int lines = (P.ny + XW - 1) / XW;
        const int seg = pick_seg_x(P.nx, lines, num_sms(), NMSDT_X_MINBLOCKS, 2.5);
        sweep_dispatch(false, 0, mode, lim, dim3(lines, (P.nx + seg - 1) / seg), s, pdl, P, qin, tm_in, qout, dtp, ctl, seg, end_step && mode >= MODE_TRAIL ? 1 : 0);
    } else {
        const int lines = (P.nx + YT - 1) / YT;
        const int seg = pick_seg(P.ny, 128, 4, 1.5, lines, num_sms(), NMSDT_Y_MINBLOCKS, 1.3);
        sweep_dispatch(false, 1, mode, lim, dim3(lines, (P.ny + seg - 1) / seg), s, pdl, P, qin, tm_in, qout, dtp, ctl, seg, end_step && mode >= MODE_TRAIL ? 1 : 0);
    }
}

// launch geometry of a fused sweep (sim_sweep_geometry): cells a block marches over, ramp-up cells in front, number of blocks
void sweep_geometry(const Params& P, int dir, int* seg, int* ramp, long long* nblocks)
{
    if (dir == 0) {
        const int lines = (P.ny + XW - 1) / XW;
        *seg = pick_seg_x(P.nx, lines, num_sms(), NMSDT_X_MINBLOCKS, 2.5); *ramp = XRAMP;
        *nblocks = (long long)lines * ((P.nx + *seg - 1) / *seg);
    } else {
        const int lines = (P.nx + YT - 1) / YT;
        *seg = pick_seg(P.ny, 128, 4, 1.5, lines, num_sms(), NMSDT_Y_MINBLOCKS, 1.3); *ramp = 4;
        *nblocks = (long long)lines * ((P.ny + *seg - 1) / *seg);
    }
}

void launch_source_fast(const Params& P, double* q, const double* dtp, cudaStream_t s)
{
    dim3 grid((P.nx + 127) / 128, P.ny);
    k_source_fast<<<grid, 128, 0, s>>>(P, q, dtp);
}

void launch_ctl(const Params& P, Ctl* ctl, int advance, cudaStream_t s, bool pdl) { launch_k(k_ctl, dim3(1), dim3(1), 0, s, pdl, P, ctl, advance); }

double host_tsafe(double tau, double Cpre, double Ta, double theta0) { return tsafe_for(tau, Cpre, Ta, theta0); }

} // namespace nmsdt
