/*
 * nmsdt_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded-by-default CPU implementation (fp64) of the per-time-step
 * finite-volume update of the 2D diffuse-interface two-fluid reactive Euler model of
 * Mi et al., arXiv:1905.05727 (PAPER.md, "P:n" = line n).  It is written from the paper
 * and from the readings listed in DESIGN.md ("R1".."R22"); it shares no code, header,
 * table or helper with the CUDA path under paper_1905_05727_b200/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call anything in this directory.
 *
 * Parity pins (tests/test_oracle_*.py): see DESIGN.md "Oracle pins".  Functions whose
 * behaviour is not pinned by anything outside this file say "parity unpinned" below.
 *
 * State vector per cell (Eq. 1), SoA, fp64:
 *   q0 = z1*rho1, q1 = z2*rho2, q2 = rho*u, q3 = rho*v, q4 = rho*E, q5 = z1, q6 = z2*rho2*lambda
 * Primitive vector W = (rho1, rho2, u, v, p, z1, lambda).
 */
#ifndef NMSDT_ORACLE_H
#define NMSDT_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc orc_t;

enum { ORC_BC_TRANSMISSIVE = 0, ORC_BC_PERIODIC = 1, ORC_BC_REFLECTIVE = 2, ORC_BC_INFLOW_FIXED = 3 };
enum { ORC_LIM_MINMOD = 0, ORC_LIM_MC = 1 };

typedef struct {
    int nx, ny;
    double dx, dy;
    int bc_xlo, bc_xhi, bc_ylo, bc_yhi;
    double cfl;
    int limiter;
} orc_grid_t;

/* Table I, Table II, T_ref,2 = 0 K */
typedef struct {
    double gamma1, cv1;
    double Gamma2, A, B, C, D, rho02, cv2, Tref2;
    double z_min;
} orc_eos_t;

/* Table III + sub-stepping rule R13 */
typedef struct {
    double Ta, Cpre, Q;
    int reactive;
    int max_substeps;
    double substep_theta;
} orc_kin_t;

typedef struct { double x, y, r; } orc_cavity_t; /* cell units */

typedef struct {
    double p_shock;
    int shock_cells;
    double p0, rho1_0, rho2_0;
    double interface_width;
    const orc_cavity_t* cav; int ncav;          /* explicit list ... */
    unsigned long long seed;                     /* ... or seeded generator (phi > 0) */
    double phi, dmin, dmax, min_gap;
    int x_lo, x_hi;
    int lattice; double lattice_d, lattice_spacing; /* ... or square lattice */
} orc_init_t;

typedef struct {
    double t; long long step; double dt_last, smax;
    double M2r, M2tot0, burned_mass, rate_inst;
    double mass1, mass2, momx, momy, energy;
    int bad_state;
} orc_diag_t;

/* ---- simulation object --------------------------------------------------------- */
int  orc_create(const orc_grid_t*, const orc_eos_t*, const orc_kin_t*, orc_t** out);
void orc_destroy(orc_t*);
void orc_set_threads(orc_t*, int nthreads);        /* OpenMP over rows only; results bit-identical */
int  orc_init(orc_t*, const orc_init_t*);
int  orc_init_fields(orc_t*, const double* const q[7]);
int  orc_cfl_dt(orc_t*, double* dt_out);
int  orc_step(orc_t*, int n);
int  orc_step_dt(orc_t*, int n, double dt);
int  orc_diagnostics(orc_t*, orc_diag_t* out);
int  orc_read_field(orc_t*, int field_id, double* out);
int  orc_get_cavities(orc_t*, orc_cavity_t* out, int cap, int* n);
long long orc_fallback_count(orc_t*);              /* number of first-order fallbacks so far */

/* ---- post-processing of the paper's figures (readings R23-R26 of DESIGN.md) --------------
 * orc_profiles: Eq. 9-11 by the midpoint rule on the uniform grid, plain sequential sums over j:
 *   pbar_i = (1/ny) sum_j p_ij,  rhobar_i = (1/ny) sum_j rho_ij,  ubar_i = sum_j (rho u)_ij / sum_j rho_ij,
 *   and the leading-shock position of Appendix C: x_s = dx * (1 + max{i : pbar_i >= p_front}), 0 if none
 *   (the paper's p_front is 1.01 p0).  Any output pointer may be NULL.
 * orc_qdot_pdf: Eq. 14-16: qdot = q6 C exp(-Ta/T2) Q [W/m^3] (0 when inert or T2 <= 0),
 *   n = log10(qdot / 1e9), bin b = floor((n - n_lo)/dn) counted iff 0 <= b < nbins; mass[b] += q1 dx dy (the mass of NM
 *   in the cell), count[b] += 1.  Eq. 16's f = mass / (M2tot0 dn) is left to the caller.
 * orc_shock_kinematics: Eq. C1-C2 on samples (t_k, xs_k) with x_s(t) interpolated linearly between
 *   samples: us_k = [x_s(t_k + dtau/2) - x_s(t_k - dtau/2)]/dtau, as_k = [x_s(t_k + dtau) - 2 x_s(t_k) + x_s(t_k - dtau)]/dtau^2
 *   (C1 substituted into C2); NaN where the window leaves [t_0, t_{n-1}]. */
int  orc_profiles(orc_t*, double p_front, double* pbar, double* rhobar, double* ubar, double* xs_out);
int  orc_qdot_pdf(orc_t*, double n_lo, double dn, int nbins, double* mass, long long* count);
int  orc_shock_kinematics(const double* t, const double* xs, int n, double dtau, double* us, double* as);

/* ---- pieces of the step, exposed so that tests can pin them one by one ----------- */
int  orc_halo(orc_t*, int dir);                    /* fill ghosts for a sweep in dir (0 = x, 1 = y) */
int  orc_sweep(orc_t*, int dir, double dt);        /* halo + one directional MUSCL-Hancock/HLLC sweep */
int  orc_source(orc_t*, double tau);               /* Arrhenius source over tau on every cell */

/* ---- pointwise model functions -------------------------------------------------- */
double orc_pref2(const orc_eos_t*, double rho2);                       /* Eq. 3 */
double orc_eref2(const orc_eos_t*, double rho2);                       /* Eq. 4 */
double orc_e2(const orc_eos_t*, double rho2, double p);                /* Eq. 2 solved for e2 */
double orc_T2(const orc_eos_t*, double rho2, double p);                /* Eq. 5, i = 2 */
double orc_T1(const orc_eos_t*, double rho1, double p);                /* Eq. 5, i = 1 */
double orc_mix_rhoe(const orc_eos_t*, double z1, double rho2, double p);   /* P:58 + Eq. 2 */
double orc_mix_p(const orc_eos_t*, double z1, double rho2, double rhoe);
double orc_mix_rhoc2(const orc_eos_t*, double z1, double rho2, double p);  /* R10 */
void   orc_cons_to_prim(const orc_eos_t*, const double q[7], double W[7], double* c, double* T2);
void   orc_prim_to_cons(const orc_eos_t*, const double W[7], double q[7]);
/* HLLC flux and face velocity for a face with normal along x (R9, O4.3-5) */
void   orc_hllc(const orc_eos_t*, const double WL[7], const double WR[7], double F[7], double* uface);
/* one-cell source step over tau (O5); returns number of RK4 sub-steps taken */
int    orc_source_cell(const orc_eos_t*, const orc_kin_t*, double q[7], double tau);
/* neat-NM shock Hugoniot from (p0, rho2_0) to p_s: out = {rho_s, U_s, u_p, T2_s, rho1_s} */
int    orc_hugoniot(const orc_eos_t*, double p0, double rho1_0, double rho2_0, double p_s, double out[5]);
/* seeded cavity generator (R16); returns count */
int    orc_gen_cavities(unsigned long long seed, double phi, double dmin, double dmax, double min_gap,
                        int x_lo, int x_hi, int ny, int periodic_y, orc_cavity_t* out, int cap);
double orc_limiter(int kind, double a, double b);

#ifdef __cplusplus
}
#endif
#endif
