/*
 * nmsdt_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see nmsdt_oracle.h).
 *
 * Plain fp64 CPU oracle of the per-step update of Mi et al., arXiv:1905.05727.
 * Every function cites the passage of PAPER.md ("P:n") or the DESIGN.md reading ("Rn")
 * it follows.  The algorithm is written line by line in the paper's order:
 *   Strang splitting hydro/reaction  ->  orc_step
 *   MUSCL-Hancock + slope limiter + HLLC per direction  ->  sweep_line
 *   single-step Arrhenius (Eq. 6)  ->  orc_source_cell
 *   Cochran-Chan / ideal gas + isobaric mixture (Eq. 2-5)  ->  orc_mix_*
 * No blocking, fusion or reordering.  Build with -O2 -ffp-contract=off (no FMA contraction)
 * so that every decision is taken on exactly rounded +,-,*,/ results.
 *
 * Pins: tests/test_oracle_eos.py, test_oracle_riemann.py, test_oracle_invariants.py,
 * test_oracle_source.py, test_oracle_init.py, test_oracle_sdt.py.
 * "parity unpinned": 2D cavity-collapse fields (paper prints no field values).
 */
#include "nmsdt_oracle.h"

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int NG = 2;           /* stencil radius i-2..i+2 (MUSCL-Hancock) */
constexpr double C_FLOOR2 = 1.0; /* R10: sound-speed floor (1 m/s)^2 */

inline double clampd(double x, double lo, double hi) { return x < lo ? lo : (x > hi ? hi : x); }

} // namespace

struct orc {
    orc_grid_t g;
    orc_eos_t e;
    orc_kin_t k;
    int sx, sy;                         /* padded sizes nx+4, ny+4 */
    std::vector<double> q[7];
    std::vector<double> inflow[7];      /* ORC_BC_INFLOW_FIXED state per row (captured at init) */
    std::vector<orc_cavity_t> cav;
    double t = 0.0, dt_last = 0.0, M2tot0 = 0.0;
    long long step = 0;
    long long fallbacks = 0;
    int nthreads = 1;
    bool inited = false;
    inline size_t idx(int i, int j) const { return (size_t)(j + NG) * sx + (size_t)(i + NG); }
};

/* =============================== EOS ================================== */

extern "C" double orc_pref2(const orc_eos_t* e, double rho2)
{   /* Eq. 3: (rho0/rho)^(-C) = x^C with x = rho/rho0 */
    double x = rho2 / e->rho02;
    return e->A * std::pow(x, e->C) - e->B * std::pow(x, e->D);
}

extern "C" double orc_eref2(const orc_eos_t* e, double rho2)
{   /* Eq. 4: (rho0/rho)^(1-C) = x^(C-1) */
    double x = rho2 / e->rho02;
    return -e->A / (e->rho02 * (1.0 - e->C)) * (std::pow(x, e->C - 1.0) - 1.0)
           + e->B / (e->rho02 * (1.0 - e->D)) * (std::pow(x, e->D - 1.0) - 1.0);
}

static inline double rho_eref2(const orc_eos_t* e, double rho2)
{   /* rho2 * Eq. 4: -A/(1-C) (x^C - x) + B/(1-D) (x^D - x)   (O2) */
    double x = rho2 / e->rho02;
    return -e->A / (1.0 - e->C) * (std::pow(x, e->C) - x) + e->B / (1.0 - e->D) * (std::pow(x, e->D) - x);
}

extern "C" double orc_e2(const orc_eos_t* e, double rho2, double p)
{   /* Eq. 2 solved for e2 */
    return orc_eref2(e, rho2) + (p - orc_pref2(e, rho2)) / (rho2 * e->Gamma2);
}

extern "C" double orc_T2(const orc_eos_t* e, double rho2, double p)
{   /* Eq. 5 with constant Gamma2, cv2, T_ref,2 = 0 K */
    return e->Tref2 + (p - orc_pref2(e, rho2)) / (rho2 * e->Gamma2 * e->cv2);
}

extern "C" double orc_T1(const orc_eos_t* e, double rho1, double p)
{   /* Eq. 5 with p_ref,1 = 0, T_ref,1 = 0, Gamma1 = gamma1 - 1 */
    return p / (rho1 * (e->gamma1 - 1.0) * e->cv1);
}

extern "C" double orc_mix_rhoe(const orc_eos_t* e, double z1, double rho2, double p)
{   /* rho e = z1 rho1 e1 + z2 rho2 e2; rho1 e1 = p/(gamma1-1); Eq. 2 for phase 2 */
    double z2 = 1.0 - z1;
    double G1 = e->gamma1 - 1.0;
    return z1 * p / G1 + z2 * (rho_eref2(e, rho2) + (p - orc_pref2(e, rho2)) / e->Gamma2);
}

extern "C" double orc_mix_p(const orc_eos_t* e, double z1, double rho2, double rhoe)
{   /* inverse of orc_mix_rhoe: p = [rho e - z2 (rho2 e_ref2 - p_ref2/Gamma2)] / xi   (O2) */
    double z2 = 1.0 - z1;
    double G1 = e->gamma1 - 1.0;
    double xi = z1 / G1 + z2 / e->Gamma2;
    return (rhoe - z2 * (rho_eref2(e, rho2) - orc_pref2(e, rho2) / e->Gamma2)) / xi;
}

extern "C" double orc_mix_rhoc2(const orc_eos_t* e, double z1, double rho2, double p)
{   /* R10: frozen mixture sound speed, rho c^2 = [z1 gamma1 p/G1 + z2 rho2 c2^2/G2]/xi, with the
       Mie-Grueneisen phase sound speed rho2 c2^2 = (A C x^C - B D x^D) + (G2+1)(p - p_ref2). */
    double z2 = 1.0 - z1;
    double G1 = e->gamma1 - 1.0;
    double xi = z1 / G1 + z2 / e->Gamma2;
    double x = rho2 / e->rho02;
    double xC = std::pow(x, e->C), xD = std::pow(x, e->D);
    double pref = e->A * xC - e->B * xD;
    double rho2c22 = (e->A * e->C * xC - e->B * e->D * xD) + (e->Gamma2 + 1.0) * (p - pref);
    return (z1 * e->gamma1 * p / G1 + z2 * rho2c22 / e->Gamma2) / xi;
}

extern "C" void orc_cons_to_prim(const orc_eos_t* e, const double q[7], double W[7], double* c, double* T2)
{   /* O3 */
    double rho = q[0] + q[1];
    double u = q[2] / rho, v = q[3] / rho;
    double z1 = clampd(q[5], e->z_min, 1.0 - e->z_min);
    double z2 = 1.0 - z1;
    double rho1 = q[0] / z1, rho2 = q[1] / z2;
    double rhoe = q[4] - 0.5 * (q[2] * q[2] + q[3] * q[3]) / rho;
    double p = orc_mix_p(e, z1, rho2, rhoe);
    double lam = clampd(q[6] / q[1], 0.0, 1.0);
    W[0] = rho1; W[1] = rho2; W[2] = u; W[3] = v; W[4] = p; W[5] = z1; W[6] = lam;
    if (c) {
        double c2 = orc_mix_rhoc2(e, z1, rho2, p) / rho;
        *c = std::sqrt(c2 > C_FLOOR2 ? c2 : C_FLOOR2);
    }
    if (T2) *T2 = orc_T2(e, rho2, p);
}

extern "C" void orc_prim_to_cons(const orc_eos_t* e, const double W[7], double q[7])
{
    double z1 = W[5], z2 = 1.0 - z1;
    double rho = z1 * W[0] + z2 * W[1];
    q[0] = z1 * W[0];
    q[1] = z2 * W[1];
    q[2] = rho * W[2];
    q[3] = rho * W[3];
    q[4] = orc_mix_rhoe(e, z1, W[1], W[4]) + 0.5 * rho * (W[2] * W[2] + W[3] * W[3]);
    q[5] = z1;
    q[6] = q[1] * W[6];
}

/* ============================ limiter (R5) ======================================= */

extern "C" double orc_limiter(int kind, double a, double b)
{
    if (!(a * b > 0.0)) return 0.0;
    if (kind == ORC_LIM_MC) {
        double m = std::fmin(2.0 * std::fabs(a), 2.0 * std::fabs(b));
        m = std::fmin(m, 0.5 * std::fabs(a + b));
        return a > 0.0 ? m : -m;
    }
    return std::fabs(a) < std::fabs(b) ? a : b; /* minmod */
}

/* ============================ HLLC (O4.3-5, R9) ================================== */

namespace {

struct FaceState {       /* everything HLLC needs about one side of a face */
    double U[7], F[7];
    double rho, un, p, c;
};

void face_state(const orc_eos_t* e, const double W[7], FaceState& s)
{
    double z1 = W[5], z2 = 1.0 - z1;
    double rho = z1 * W[0] + z2 * W[1];
    double u = W[2], v = W[3], p = W[4];
    double rhoE = orc_mix_rhoe(e, z1, W[1], p) + 0.5 * rho * (u * u + v * v);
    double c2 = orc_mix_rhoc2(e, z1, W[1], p) / rho;
    s.rho = rho; s.un = u; s.p = p;
    s.c = std::sqrt(c2 > C_FLOOR2 ? c2 : C_FLOOR2);
    s.U[0] = z1 * W[0]; s.U[1] = z2 * W[1]; s.U[2] = rho * u; s.U[3] = rho * v; s.U[4] = rhoE;
    s.U[5] = z1;        s.U[6] = s.U[1] * W[6];
    s.F[0] = s.U[0] * u; s.F[1] = s.U[1] * u; s.F[2] = rho * u * u + p; s.F[3] = rho * u * v;
    s.F[4] = (rhoE + p) * u; s.F[5] = z1 * u; s.F[6] = s.U[6] * u;
}

void hllc_flux(const FaceState& L, const FaceState& R, double F[7], double* uface)
{
    /* R9: Davis wave-speed estimates */
    double SL = std::fmin(L.un - L.c, R.un - R.c);
    double SR = std::fmax(L.un + L.c, R.un + R.c);
    double Sstar = (R.p - L.p + L.rho * L.un * (SL - L.un) - R.rho * R.un * (SR - R.un))
                   / (L.rho * (SL - L.un) - R.rho * (SR - R.un));
    if (SL >= 0.0) {
        for (int k = 0; k < 7; ++k) F[k] = L.F[k];
        *uface = L.un;
        return;
    }
    if (!(SR > 0.0)) {
        for (int k = 0; k < 7; ++k) F[k] = R.F[k];
        *uface = R.un;
        return;
    }
    const FaceState& K = (Sstar >= 0.0) ? L : R;
    double SK = (Sstar >= 0.0) ? SL : SR;
    double chi = (SK - K.un) / (SK - Sstar);
    double Us[7];
    for (int k = 0; k < 7; ++k) Us[k] = chi * K.U[k];
    Us[2] = K.rho * chi * Sstar;
    double EK = K.U[4] / K.rho; /* specific total energy */
    Us[4] = K.rho * chi * (EK + (Sstar - K.un) * (Sstar + K.p / (K.rho * (SK - K.un))));
    for (int k = 0; k < 7; ++k) F[k] = K.F[k] + SK * (Us[k] - K.U[k]);
    *uface = K.un + SK * (chi - 1.0);
}

} // namespace

extern "C" void orc_hllc(const orc_eos_t* e, const double WL[7], const double WR[7], double F[7], double* uface)
{
    FaceState L, R;
    face_state(e, WL, L);
    face_state(e, WR, R);
    hllc_flux(L, R, F, uface);
}

/* ============================ source step (O5, Eq. 6) ============================ */

extern "C" int orc_source_cell(const orc_eos_t* e, const orc_kin_t* k, double q[7], double tau)
{
    if (!k->reactive) return 0;
    double W[7], T0;
    orc_cons_to_prim(e, q, W, nullptr, &T0);
    double z1 = W[5], z2 = 1.0 - z1, lam0 = W[6];
    double G1 = e->gamma1 - 1.0;
    double xi = z1 / G1 + z2 / e->Gamma2;
    /* hydrodynamic variables frozen, p linear in rho e  =>  T2(lam) = T0 + beta (lam0 - lam) */
    double beta = z2 * k->Q / (xi * e->Gamma2 * e->cv2);
    /* R13: sub-step count from exactly rounded operations only */
    double Tub = T0 + beta * lam0;
    int nsub = 1;
    if (Tub > 0.0) {
        double y = k->Ta / Tub;
        double g = 1.0 / (1.0 + y + y * y / 2.0 + y * y * y / 6.0);   /* >= exp(-y) */
        double theta = tau * k->Cpre * g;
        double r = std::floor(theta / k->substep_theta);
        nsub = (r >= (double)(k->max_substeps - 1)) ? k->max_substeps : 1 + (int)r;
    }
    auto f = [&](double l) {   /* Eq. 6: K = -lambda C exp(-Ta/T2) */
        double T = T0 + beta * (lam0 - l);
        return T > 0.0 ? -l * k->Cpre * std::exp(-k->Ta / T) : 0.0;
    };
    double h = tau / (double)nsub;
    double lam = lam0;
    for (int s = 0; s < nsub; ++s) {  /* classic RK4 */
        double k1 = f(lam);
        double k2 = f(lam + 0.5 * h * k1);
        double k3 = f(lam + 0.5 * h * k2);
        double k4 = f(lam + h * k3);
        lam = lam + h / 6.0 * (k1 + 2.0 * k2 + 2.0 * k3 + k4);
    }
    double lam1 = clampd(lam, 0.0, lam0);
    q[6] = q[1] * lam1;
    q[4] = q[4] + q[1] * k->Q * (lam0 - lam1);   /* Eq. 1 energy source -z2 rho2 K Q */
    return nsub;
}

/* ============================ Hugoniot init (O7) ========================== */

extern "C" int orc_hugoniot(const orc_eos_t* e, double p0, double rho1_0, double rho2_0, double ps, double out[5])
{
    double e0 = orc_e2(e, rho2_0, p0);
    double v0 = 1.0 / rho2_0;
    auto f = [&](double rho) { return orc_e2(e, rho, ps) - e0 - 0.5 * (ps + p0) * (v0 - 1.0 / rho); };
    double lo = rho2_0 * (1.0 + 1e-12), hi = rho2_0 * 1.5;
    if (!(ps > p0) || !(f(lo) > 0.0)) return -1;
    int guard = 0;
    while (f(hi) > 0.0) { hi *= 1.5; if (++guard > 40) return -1; }
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (f(mid) > 0.0) lo = mid; else hi = mid;
    }
    double rs = 0.5 * (lo + hi);
    double up = std::sqrt((ps - p0) * (v0 - 1.0 / rs));
    double Us = up / (1.0 - rho2_0 / rs);
    double g = e->gamma1;
    out[0] = rs; out[1] = Us; out[2] = up; out[3] = orc_T2(e, rs, ps);
    out[4] = rho1_0 * ((g + 1.0) * ps + (g - 1.0) * p0) / ((g - 1.0) * ps + (g + 1.0) * p0); /* air shock Hugoniot */
    return 0;
}

/* ============================ cavity generator (R16) ============================= */

namespace {

inline uint64_t mix64(uint64_t x)
{   /* splitmix64 finaliser: counter-based, the CUDA side implements the same function */
    x += 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}
inline uint64_t rnd(uint64_t seed, uint64_t k, uint64_t s) { return mix64(mix64(seed) + 4ULL * k + s); }
inline uint64_t mulhi(uint64_t a, uint64_t b) { return (uint64_t)(((unsigned __int128)a * b) >> 64); }

} // namespace

extern "C" int orc_gen_cavities(unsigned long long seed, double phi, double dmin, double dmax, double min_gap,
                                int x_lo, int x_hi, int ny, int periodic_y, orc_cavity_t* out, int cap)
{
    /* fixed point: 1/256 cell.  Sequential greedy rejection sampling. */
    const int64_t Rmin = (int64_t)std::llround(dmin * 128.0), Rmax = (int64_t)std::llround(dmax * 128.0);
    const int64_t G = (int64_t)std::llround(min_gap * 256.0);
    const int64_t H = (int64_t)ny * 256;
    const int64_t target = (int64_t)std::floor(phi * (double)(x_hi - x_lo) * (double)ny * 65536.0 / 3.14159265358979323846);
    if (Rmin <= 0 || Rmax < Rmin || x_hi <= x_lo || ny <= 0) return -1;
    /* candidate budget: 256 candidates per cavity of the target.  The paper's densest case (phi = 8 %, centre spacing
       2.5 d_c) fills 0.50 of the plane with exclusion disks, close to the ~0.547 jamming limit of random
       sequential placement, and needs ~40 candidates per cavity; a target beyond the jamming limit ends here. */
    const int64_t max_cand = 256 * (target / (Rmin * Rmin) + 1) + 1024;
    std::vector<int64_t> X, Y, R;
    int64_t sum = 0;
    for (int64_t k = 0; k < max_cand && sum < target; ++k) {
        int64_t Rk = Rmin + (int64_t)mulhi(rnd(seed, k, 2), (uint64_t)(Rmax - Rmin + 1));
        int64_t xlo = (int64_t)x_lo * 256 + Rk, xhi = (int64_t)x_hi * 256 - Rk;
        if (xhi < xlo) continue;
        int64_t Xk = xlo + (int64_t)mulhi(rnd(seed, k, 0), (uint64_t)(xhi - xlo + 1));
        int64_t Yk;
        if (periodic_y) Yk = (int64_t)mulhi(rnd(seed, k, 1), (uint64_t)H);
        else {
            int64_t ylo = Rk, yhi = H - Rk;
            if (yhi < ylo) continue;
            Yk = ylo + (int64_t)mulhi(rnd(seed, k, 1), (uint64_t)(yhi - ylo + 1));
        }
        bool ok = true;
        for (size_t j = 0; j < X.size(); ++j) {
            int64_t ddx = Xk - X[j];
            int64_t ddy = Yk > Y[j] ? Yk - Y[j] : Y[j] - Yk;
            if (periodic_y && 2 * ddy > H) ddy = H - ddy;
            int64_t lim = Rk + R[j] + G;
            if (ddx * ddx + ddy * ddy < lim * lim) { ok = false; break; }
        }
        if (!ok) continue;
        X.push_back(Xk); Y.push_back(Yk); R.push_back(Rk);
        sum += Rk * Rk;
    }
    int n = (int)X.size();
    for (int j = 0; j < n && j < cap; ++j) {
        out[j].x = (double)X[j] / 256.0; out[j].y = (double)Y[j] / 256.0; out[j].r = (double)R[j] / 256.0;
    }
    return n;
}

/* ============================ simulation object ================================== */

extern "C" int orc_create(const orc_grid_t* g, const orc_eos_t* e, const orc_kin_t* k, orc_t** out)
{
    if (!g || !e || !k || !out || g->nx < 1 || g->ny < 1 || !(g->dx > 0) || !(g->dy > 0)) return -1;
    if (g->bc_xhi == ORC_BC_INFLOW_FIXED || g->bc_ylo == ORC_BC_INFLOW_FIXED || g->bc_yhi == ORC_BC_INFLOW_FIXED) return -1;
    if ((g->bc_xlo == ORC_BC_PERIODIC) != (g->bc_xhi == ORC_BC_PERIODIC)) return -1;
    if ((g->bc_ylo == ORC_BC_PERIODIC) != (g->bc_yhi == ORC_BC_PERIODIC)) return -1;
    orc* s = new orc();
    s->g = *g; s->e = *e; s->k = *k;
    s->sx = g->nx + 2 * NG; s->sy = g->ny + 2 * NG;
    for (int f = 0; f < 7; ++f) { s->q[f].assign((size_t)s->sx * s->sy, 0.0); s->inflow[f].assign(g->ny, 0.0); }
    *out = s;
    return 0;
}

extern "C" void orc_destroy(orc_t* s) { delete s; }

extern "C" void orc_set_threads(orc_t* s, int n) { s->nthreads = n < 1 ? 1 : n; }

extern "C" long long orc_fallback_count(orc_t* s) { return s->fallbacks; }

static void finish_init(orc* s)
{
    for (int f = 0; f < 7; ++f)
        for (int j = 0; j < s->g.ny; ++j) s->inflow[f][j] = s->q[f][s->idx(0, j)];
    s->t = 0.0; s->step = 0; s->dt_last = 0.0; s->fallbacks = 0;
    double M = 0.0;
    for (int j = 0; j < s->g.ny; ++j)
        for (int i = 0; i < s->g.nx; ++i) M += s->q[6][s->idx(i, j)];
    s->M2tot0 = M * s->g.dx * s->g.dy;
    s->inited = true;
}

extern "C" int orc_init_fields(orc_t* s, const double* const q[7])
{
    if (!s || !q) return -1;
    for (int f = 0; f < 7; ++f)
        for (int j = 0; j < s->g.ny; ++j)
            for (int i = 0; i < s->g.nx; ++i) s->q[f][s->idx(i, j)] = q[f][(size_t)j * s->g.nx + i];
    /* R27: the stored volume fraction of every state the scheme holds lies in [z_min, 1 - z_min] -- O7 paints it
       there, O4.6 clamps each update, O3 clamps at each primitive recovery -- so a caller's state is brought to the same
       invariant on entry; otherwise O4.6 would use the raw value in the z1 (u* difference) term of the first sweep only. */
    for (int j = 0; j < s->g.ny; ++j)
        for (int i = 0; i < s->g.nx; ++i) {
            double& z = s->q[5][s->idx(i, j)];
            z = clampd(z, s->e.z_min, 1.0 - s->e.z_min);
        }
    s->cav.clear();
    finish_init(s);
    return 0;
}

extern "C" int orc_init(orc_t* s, const orc_init_t* in)
{   /* O7 */
    if (!s || !in) return -1;
    const orc_eos_t* e = &s->e;
    const int nx = s->g.nx, ny = s->g.ny;
    const bool per_y = s->g.bc_ylo == ORC_BC_PERIODIC;
    /* cavity list */
    s->cav.clear();
    if (in->cav && in->ncav > 0) s->cav.assign(in->cav, in->cav + in->ncav);
    else if (in->lattice) {   /* Eq. 7 geometry, R20: centres x_lo + s/2 + s i, s/2 + s j */
        double sp = in->lattice_spacing, r = 0.5 * in->lattice_d;
        for (int jj = 0; sp * (jj + 1) <= (double)ny; ++jj)
            for (int ii = 0; in->x_lo + sp * (ii + 1) <= (double)in->x_hi; ++ii)
                s->cav.push_back({in->x_lo + 0.5 * sp + sp * ii, 0.5 * sp + sp * jj, r});
    } else if (in->phi > 0.0) {
        std::vector<orc_cavity_t> tmp(1 << 20);
        int n = orc_gen_cavities(in->seed, in->phi, in->dmin, in->dmax, in->min_gap, in->x_lo, in->x_hi, ny,
                                 per_y ? 1 : 0, tmp.data(), (int)tmp.size());
        if (n < 0 || n > (int)tmp.size()) return -1;
        s->cav.assign(tmp.begin(), tmp.begin() + n);
    }
    /* profile = max_k 1/2 [1 - tanh((d_k - R_k)/h)], h = interface_width/2 (R15); exactly 0 beyond 20 h */
    std::vector<double> prof((size_t)nx * ny, 0.0);
    const double h = 0.5 * in->interface_width;
    for (const orc_cavity_t& c : s->cav) {
        double reach = c.r + 20.0 * h + 1.0;
        int i0 = (int)std::floor(c.x - reach), i1 = (int)std::ceil(c.x + reach);
        int j0 = (int)std::floor(c.y - reach), j1 = (int)std::ceil(c.y + reach);
        for (int jj = j0; jj <= j1; ++jj) {
            int j = jj;
            if (per_y) j = ((jj % ny) + ny) % ny;   /* rows may be visited twice: max is idempotent */
            else if (jj < 0 || jj >= ny) continue;
            for (int i = std::max(i0, 0); i <= std::min(i1, nx - 1); ++i) {
                double ddx = (i + 0.5) - c.x;
                double ddy = std::fabs((j + 0.5) - c.y);
                if (per_y && ddy > 0.5 * ny) ddy = ny - ddy;     /* minimum image */
                double d = std::sqrt(ddx * ddx + ddy * ddy);
                double sarg = (d - c.r) / h;
                double val = sarg >= 20.0 ? 0.0 : 1.0 / (1.0 + std::exp(2.0 * sarg));   /* = 1/2 [1 - tanh(s)], well conditioned in the tail */
                double& pr = prof[(size_t)j * nx + i];
                if (val > pr) pr = val;
            }
        }
    }
    double hug[5] = {0, 0, 0, 0, 0};
    if (in->shock_cells > 0 && orc_hugoniot(e, in->p0, in->rho1_0, in->rho2_0, in->p_shock, hug) != 0) return -1;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            double W[7], q[7];
            if (i < in->shock_cells) {   /* shocked slab: neat-NM Hugoniot state, lambda = 0 */
                W[0] = hug[4]; W[1] = hug[0]; W[2] = hug[2]; W[3] = 0.0; W[4] = in->p_shock;
                W[5] = e->z_min; W[6] = 0.0;
            } else {                     /* ambient, lambda = 1 */
                W[0] = in->rho1_0; W[1] = in->rho2_0; W[2] = 0.0; W[3] = 0.0; W[4] = in->p0;
                W[5] = e->z_min + (1.0 - 2.0 * e->z_min) * prof[(size_t)j * nx + i]; W[6] = 1.0;
            }
            orc_prim_to_cons(e, W, q);
            for (int f = 0; f < 7; ++f) s->q[f][s->idx(i, j)] = q[f];
        }
    finish_init(s);
    return 0;
}

extern "C" int orc_get_cavities(orc_t* s, orc_cavity_t* out, int cap, int* n)
{
    if (!s || !n) return -1;
    *n = (int)s->cav.size();
    for (int j = 0; j < *n && j < cap; ++j) out[j] = s->cav[j];
    return 0;
}

/* ============================ halo (a2) ============================= */

extern "C" int orc_halo(orc_t* s, int dir)
{
    const int nx = s->g.nx, ny = s->g.ny;
    if (dir == 0) {
        for (int j = 0; j < ny; ++j)
            for (int f = 0; f < 7; ++f) {
                std::vector<double>& a = s->q[f];
                for (int m = 1; m <= NG; ++m) {
                    /* low side, ghost i = -m */
                    double v;
                    switch (s->g.bc_xlo) {
                        case ORC_BC_PERIODIC:     v = a[s->idx(((nx - m) % nx + nx) % nx, j)]; break;
                        case ORC_BC_REFLECTIVE:   v = a[s->idx(m - 1, j)]; if (f == 2) v = -v; break;
                        case ORC_BC_INFLOW_FIXED: v = s->inflow[f][j]; break;
                        default:                  v = a[s->idx(0, j)]; break;    /* zero-gradient (R12) */
                    }
                    a[s->idx(-m, j)] = v;
                    /* high side, ghost i = nx-1+m */
                    switch (s->g.bc_xhi) {
                        case ORC_BC_PERIODIC:   v = a[s->idx((m - 1) % nx, j)]; break;
                        case ORC_BC_REFLECTIVE: v = a[s->idx(nx - m, j)]; if (f == 2) v = -v; break;
                        default:                v = a[s->idx(nx - 1, j)]; break;
                    }
                    a[s->idx(nx - 1 + m, j)] = v;
                }
            }
    } else {
        for (int f = 0; f < 7; ++f) {
            std::vector<double>& a = s->q[f];
            for (int m = 1; m <= NG; ++m)
                for (int i = 0; i < nx; ++i) {
                    double v;
                    switch (s->g.bc_ylo) {
                        case ORC_BC_PERIODIC:   v = a[s->idx(i, ((ny - m) % ny + ny) % ny)]; break;
                        case ORC_BC_REFLECTIVE: v = a[s->idx(i, m - 1)]; if (f == 3) v = -v; break;
                        default:                v = a[s->idx(i, 0)]; break;
                    }
                    a[s->idx(i, -m)] = v;
                    switch (s->g.bc_yhi) {
                        case ORC_BC_PERIODIC:   v = a[s->idx(i, (m - 1) % ny)]; break;
                        case ORC_BC_REFLECTIVE: v = a[s->idx(i, ny - m)]; if (f == 3) v = -v; break;
                        default:                v = a[s->idx(i, ny - 1)]; break;
                    }
                    a[s->idx(i, ny - 1 + m)] = v;
                }
        }
    }
    return 0;
}

/* ============================ directional sweep (O4) ============================= */

namespace {

/* One line of n interior cells with 2 ghosts each side.  Q[c][k]: conserved, c = 0..n+3 (cell i = c-2),
   already arranged so that component 2 is the momentum NORMAL to the faces.  Returns fallbacks. */
int sweep_line(const orc_eos_t* e, int limiter, int n, double dtdx, std::vector<double>& Q,
               std::vector<double>& Wb, std::vector<double>& WLb, std::vector<double>& WRb,
               std::vector<double>& Fb, std::vector<double>& ub)
{
    const int m = n + 4;
    int nfb = 0;
    std::vector<double> c2b(m), rb(m);
    /* O3: primitives of every cell of the line; floored c^2 for the predictor (R10) */
    for (int c = 0; c < m; ++c) {
        double* W = &Wb[(size_t)c * 7];
        orc_cons_to_prim(e, &Q[(size_t)c * 7], W, nullptr, nullptr);
        rb[c] = Q[(size_t)c * 7 + 0] + Q[(size_t)c * 7 + 1];
        double c2 = orc_mix_rhoc2(e, W[5], W[1], W[4]) / rb[c];
        c2b[c] = c2 > C_FLOOR2 ? c2 : C_FLOOR2;
    }
    const double k = 0.5 * dtdx;
    /* O4.1-2: limited slopes and Hancock half-step predictor for cells c = 1..m-2 */
    for (int c = 1; c <= m - 2; ++c) {
        const double* Wm = &Wb[(size_t)(c - 1) * 7];
        const double* W0 = &Wb[(size_t)c * 7];
        const double* Wp = &Wb[(size_t)(c + 1) * 7];
        double D[7];
        for (int q = 0; q < 7; ++q) D[q] = orc_limiter(limiter, W0[q] - Wm[q], Wp[q] - W0[q]);
        double rho = rb[c], u = W0[2], rc2 = rho * c2b[c];
        double d[7];
        d[0] = u * D[0] + W0[0] * D[2];
        d[1] = u * D[1] + W0[1] * D[2];
        d[2] = u * D[2] + D[4] / rho;
        d[3] = u * D[3];
        d[4] = u * D[4] + rc2 * D[2];
        d[5] = u * D[5];
        d[6] = u * D[6];
        double* WL = &WLb[(size_t)c * 7];
        double* WR = &WRb[(size_t)c * 7];
        for (int q = 0; q < 7; ++q) {
            WL[q] = W0[q] - 0.5 * D[q] - k * d[q];
            WR[q] = W0[q] + 0.5 * D[q] - k * d[q];
        }
        if (!(WL[0] > 0.0) || !(WL[1] > 0.0) || !(WR[0] > 0.0) || !(WR[1] > 0.0)) {   /* R17 */
            for (int q = 0; q < 7; ++q) { WL[q] = W0[q]; WR[q] = W0[q]; }
            ++nfb;
        }
    }
    /* O4.3-5: face f between cells c = f and f+1, f = 1..m-3 */
    for (int f = 1; f <= m - 3; ++f)
        orc_hllc(e, &WRb[(size_t)f * 7], &WLb[(size_t)(f + 1) * 7], &Fb[(size_t)f * 7], &ub[f]);
    /* O4.6: update interior cells c = 2..m-3 */
    for (int c = 2; c <= m - 3; ++c) {
        double* q = &Q[(size_t)c * 7];
        const double* Fp = &Fb[(size_t)c * 7];
        const double* Fm = &Fb[(size_t)(c - 1) * 7];
        double z1n = q[5];
        for (int kk = 0; kk < 7; ++kk) q[kk] = q[kk] - dtdx * (Fp[kk] - Fm[kk]);
        q[5] = q[5] + dtdx * z1n * (ub[c] - ub[c - 1]);
        q[5] = clampd(q[5], e->z_min, 1.0 - e->z_min);
    }
    return nfb;
}

} // namespace

extern "C" int orc_sweep(orc_t* s, int dir, double dt)
{
    orc_halo(s, dir);
    const int nx = s->g.nx, ny = s->g.ny;
    const int n = dir == 0 ? nx : ny;
    const int nlines = dir == 0 ? ny : nx;
    const double dtdx = dt / (dir == 0 ? s->g.dx : s->g.dy);
    const int kn = dir == 0 ? 2 : 3, kt = dir == 0 ? 3 : 2;
    long long nfb = 0;
#ifdef _OPENMP
#pragma omp parallel num_threads(s->nthreads) reduction(+ : nfb)
#endif
    {
        const int m = n + 4;
        std::vector<double> Q((size_t)m * 7), Wb((size_t)m * 7), WLb((size_t)m * 7), WRb((size_t)m * 7),
            Fb((size_t)m * 7), ub(m);
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
        for (int l = 0; l < nlines; ++l) {
            for (int c = 0; c < m; ++c) {
                size_t id = dir == 0 ? s->idx(c - NG, l) : s->idx(l, c - NG);
                double* q = &Q[(size_t)c * 7];
                q[0] = s->q[0][id]; q[1] = s->q[1][id]; q[2] = s->q[kn][id]; q[3] = s->q[kt][id];
                q[4] = s->q[4][id]; q[5] = s->q[5][id]; q[6] = s->q[6][id];
            }
            nfb += sweep_line(&s->e, s->g.limiter, n, dtdx, Q, Wb, WLb, WRb, Fb, ub);
            for (int c = NG; c < n + NG; ++c) {
                size_t id = dir == 0 ? s->idx(c - NG, l) : s->idx(l, c - NG);
                const double* q = &Q[(size_t)c * 7];
                s->q[0][id] = q[0]; s->q[1][id] = q[1]; s->q[kn][id] = q[2]; s->q[kt][id] = q[3];
                s->q[4][id] = q[4]; s->q[5][id] = q[5]; s->q[6][id] = q[6];
            }
        }
    }
    s->fallbacks += nfb;
    return 0;
}

extern "C" int orc_source(orc_t* s, double tau)
{
    if (!s->k.reactive) return 0;
    const int nx = s->g.nx, ny = s->g.ny;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(s->nthreads)
#endif
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t id = s->idx(i, j);
            double q[7];
            for (int f = 0; f < 7; ++f) q[f] = s->q[f][id];
            orc_source_cell(&s->e, &s->k, q, tau);
            s->q[4][id] = q[4];
            s->q[6][id] = q[6];
        }
    return 0;
}

/* ============================ CFL, step, diagnostics ============================= */

static double max_wavespeed(orc* s)
{   /* a7 / R11: S_max = max over cells of max(|u|,|v|) + c */
    const int nx = s->g.nx, ny = s->g.ny;
    double smax = 0.0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(s->nthreads) reduction(max : smax)
#endif
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t id = s->idx(i, j);
            double q[7], W[7], c;
            for (int f = 0; f < 7; ++f) q[f] = s->q[f][id];
            orc_cons_to_prim(&s->e, q, W, &c, nullptr);
            double a = std::fmax(std::fabs(W[2]), std::fabs(W[3])) + c;
            if (a > smax) smax = a;
        }
    return smax;
}

extern "C" int orc_cfl_dt(orc_t* s, double* dt_out)
{
    if (!s || !s->inited) return -3;
    double smax = max_wavespeed(s);
    *dt_out = s->g.cfl * std::fmin(s->g.dx, s->g.dy) / smax;
    return 0;
}

static void one_step(orc* s, double dt)
{   /* O6 / R7: even step S X Y S, odd step S Y X S (Strang) */
    orc_source(s, 0.5 * dt);
    if ((s->step & 1LL) == 0) { orc_sweep(s, 0, dt); orc_sweep(s, 1, dt); }
    else                      { orc_sweep(s, 1, dt); orc_sweep(s, 0, dt); }
    orc_source(s, 0.5 * dt);
    s->t += dt; s->dt_last = dt; s->step += 1;
}

extern "C" int orc_step(orc_t* s, int n)
{
    if (!s || !s->inited) return -3;
    for (int it = 0; it < n; ++it) {
        double dt;
        orc_cfl_dt(s, &dt);
        one_step(s, dt);
    }
    return 0;
}

extern "C" int orc_step_dt(orc_t* s, int n, double dt)
{
    if (!s || !s->inited) return -3;
    for (int it = 0; it < n; ++it) one_step(s, dt);
    return 0;
}

extern "C" int orc_diagnostics(orc_t* s, orc_diag_t* d)
{   /* a8: Eq. 12 and conservation sums; plain sequential sums */
    if (!s || !s->inited) return -3;
    const int nx = s->g.nx, ny = s->g.ny;
    const double dA = s->g.dx * s->g.dy;
    double sum[7] = {0, 0, 0, 0, 0, 0, 0}, rate = 0.0, smax = 0.0;
    int bad = 0;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t id = s->idx(i, j);
            double q[7], W[7], c, T2;
            for (int f = 0; f < 7; ++f) { q[f] = s->q[f][id]; sum[f] += q[f]; }
            orc_cons_to_prim(&s->e, q, W, &c, &T2);
            if (s->k.reactive && T2 > 0.0) rate += q[6] * s->k.Cpre * std::exp(-s->k.Ta / T2);
            double a = std::fmax(std::fabs(W[2]), std::fabs(W[3])) + c;
            if (a > smax) smax = a;
            bool ok = std::isfinite(q[0]) && std::isfinite(q[1]) && std::isfinite(q[2]) && std::isfinite(q[3])
                      && std::isfinite(q[4]) && std::isfinite(q[5]) && std::isfinite(q[6]) && q[0] > 0.0 && q[1] > 0.0;
            if (!ok) bad = 1;
        }
    d->t = s->t; d->step = s->step; d->dt_last = s->dt_last; d->smax = smax;
    d->M2r = sum[6] * dA; d->M2tot0 = s->M2tot0; d->burned_mass = s->M2tot0 - d->M2r; d->rate_inst = rate * dA;
    d->mass1 = sum[0] * dA; d->mass2 = sum[1] * dA; d->momx = sum[2] * dA; d->momy = sum[3] * dA; d->energy = sum[4] * dA;
    d->bad_state = bad;
    return 0;
}

extern "C" int orc_read_field(orc_t* s, int id, double* out)
{
    if (!s || !s->inited || !out) return -3;
    const int nx = s->g.nx, ny = s->g.ny;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t c = s->idx(i, j);
            double v;
            if (id >= 0 && id < 7) v = s->q[id][c];
            else {
                double q[7], W[7], cs, T2;
                for (int f = 0; f < 7; ++f) q[f] = s->q[f][c];
                orc_cons_to_prim(&s->e, q, W, &cs, &T2);
                switch (id) {
                    case 16: v = W[4]; break;
                    case 17: v = T2; break;
                    case 18: v = q[0] + q[1]; break;
                    case 19: v = W[2]; break;
                    case 20: v = W[3]; break;
                    case 21: v = W[6]; break;
                    case 22: v = 1.0 - W[6]; break;
                    case 23: v = W[1]; break;
                    case 24: v = cs; break;
                    case 25: v = orc_T1(&s->e, W[0], W[4]); break;
                    case 26: v = W[0]; break;
                    default: return -1;
                }
            }
            out[(size_t)j * nx + i] = v;
        }
    return 0;
}

/* ============================ post-processing ================ */

extern "C" int orc_profiles(orc_t* s, double p_front, double* pbar, double* rhobar, double* ubar, double* xs_out)
{   /* Eq. 9-11, Appendix C front position; R23, R25 */
    if (!s || !s->inited) return -3;
    const int nx = s->g.nx, ny = s->g.ny;
    int front = -1;
    for (int i = 0; i < nx; ++i) {
        double sp = 0.0, sr = 0.0, sm = 0.0;
        for (int j = 0; j < ny; ++j) {
            size_t id = s->idx(i, j);
            double q[7], W[7], c, T2;
            for (int f = 0; f < 7; ++f) q[f] = s->q[f][id];
            orc_cons_to_prim(&s->e, q, W, &c, &T2);
            sp += W[4];
            sr += q[0] + q[1];
            sm += q[2];
        }
        const double pb = sp / (double)ny;
        if (pbar) pbar[i] = pb;
        if (rhobar) rhobar[i] = sr / (double)ny;
        if (ubar) ubar[i] = sm / sr;
        if (pb >= p_front) front = i;
    }
    if (xs_out) *xs_out = s->g.dx * (double)(front + 1);
    return 0;
}

extern "C" int orc_qdot_pdf(orc_t* s, double n_lo, double dn, int nbins, double* mass, long long* count)
{   /* Eq. 14-16; R24 */
    if (!s || !s->inited || nbins < 1 || !(dn > 0.0)) return -3;
    const int nx = s->g.nx, ny = s->g.ny;
    const double dA = s->g.dx * s->g.dy;
    for (int b = 0; b < nbins; ++b) { if (mass) mass[b] = 0.0; if (count) count[b] = 0; }
    if (!s->k.reactive) return 0;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            size_t id = s->idx(i, j);
            double q[7], W[7], c, T2;
            for (int f = 0; f < 7; ++f) q[f] = s->q[f][id];
            orc_cons_to_prim(&s->e, q, W, &c, &T2);
            if (!(T2 > 0.0)) continue;
            const double qdot = q[6] * s->k.Cpre * std::exp(-s->k.Ta / T2) * s->k.Q;     /* Eq. 14, W/m^3 */
            if (!(qdot > 0.0)) continue;
            const double n = std::log10(qdot / 1e9);                                     /* Eq. 15, GW/m^3 */
            const double fb = std::floor((n - n_lo) / dn);
            if (fb < 0.0 || fb >= (double)nbins) continue;
            const int b = (int)fb;
            if (mass) mass[b] += q[1] * dA;
            if (count) count[b] += 1;
        }
    return 0;
}

static double interp_linear(const double* t, const double* x, int n, double tq, bool* ok)
{
    if (!(tq >= t[0]) || !(tq <= t[n - 1])) { *ok = false; return 0.0; }
    int k = 0;
    while (k < n - 2 && t[k + 1] < tq) ++k;                 /* t[k] <= tq <= t[k+1] */
    const double w = (tq - t[k]) / (t[k + 1] - t[k]);
    return x[k] + w * (x[k + 1] - x[k]);
}

extern "C" int orc_shock_kinematics(const double* t, const double* xs, int n, double dtau, double* us, double* as)
{   /* Eq. C1-C2; R26 */
    if (!t || !xs || n < 2 || !(dtau > 0.0)) return -1;
    const double nan = std::nan("");
    for (int k = 0; k < n; ++k) {
        bool ok = true;
        const double xp = interp_linear(t, xs, n, t[k] + 0.5 * dtau, &ok), xm = interp_linear(t, xs, n, t[k] - 0.5 * dtau, &ok);
        if (us) us[k] = ok ? (xp - xm) / dtau : nan;
        ok = true;
        const double xpp = interp_linear(t, xs, n, t[k] + dtau, &ok), xmm = interp_linear(t, xs, n, t[k] - dtau, &ok);
        if (as) as[k] = ok ? (xpp - 2.0 * xs[k] + xmm) / (dtau * dtau) : nan;
    }
    return 0;
}
