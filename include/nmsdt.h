/*
 * nmsdt.h -- C ABI of libnmsdt.so: the B200 (sm_100a) hot path of Mi et al., arXiv:1905.05727,
 * "Meso-resolved simulations of shock-to-detonation transition in nitromethane with air-filled cavities".
 *
 * What the library computes: the per-time-step finite-volume update of the 2D diffuse-interface two-fluid
 * (air cavities = phase 1, liquid nitromethane = phase 2) reactive Euler equations, Eq. 1,
 * with the Cochran-Chan / ideal-gas equations of state Eq. 2-5, single-step Arrhenius kinetics Eq. 6
 * (P:114), MUSCL-Hancock + slope limiter + HLLC with Strang splitting, in fp64, entirely in CUDA
 * kernels on one GPU.  Points the paper leaves open are fixed by the readings R1..R22 of DESIGN.md.
 *
 * Conventions
 *  - plain C; every call returns 0 on success or a negative code:
 *      SIM_ERR_ARG (-1) bad argument, SIM_ERR_CUDA (-2) CUDA runtime error, SIM_ERR_STATE (-3) not initialised,
 *      SIM_ERR_BAD (-4) non-finite or non-positive state detected on the device.
 *    sim_last_error() returns a static / handle-owned string describing the last failure.
 *  - pointers named host_* / *_out are HOST pointers owned by the caller; the library never keeps them.
 *    `device_buf` is a DEVICE pointer.  No exception crosses the ABI.
 *  - all work is enqueued on the stream given to sim_create; calls marked [sync] block on that stream,
 *    calls marked [async] return immediately (the time step dt lives in device memory, so sim_step(n)
 *    never synchronises with the host).
 *  - there is no CPU fallback: without a CUDA device sim_create fails with SIM_ERR_CUDA.
 *
 * State per cell (SoA, fp64, 7 planes), Eq. 1:
 *   q0 = z1 rho1, q1 = z2 rho2, q2 = rho u, q3 = rho v, q4 = rho E, q5 = z1, q6 = z2 rho2 lambda
 * lambda = mass fraction of UNREACTED nitromethane, 1 -> 0.
 * Device layout: each plane is (ny+4) rows of `pitch` doubles, pitch = roundup(16 + nx + 2, 16); interior
 * cell (i,j) sits at row j+2, column 16+i, so that every interior row starts 128-byte aligned; two ghost
 * rows/columns on each side are filled by the halo step.  Two such sets of 7 planes (ping-pong) plus small
 * reduction scratch make up the workspace (sim_workspace_bytes).
 */
#ifndef NMSDT_H
#define NMSDT_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sim sim_t;

enum { SIM_OK = 0, SIM_ERR_ARG = -1, SIM_ERR_CUDA = -2, SIM_ERR_STATE = -3, SIM_ERR_BAD = -4 };
/* boundary kinds (P:129 inflow/transmissive left, P:135 periodic top/bottom; R12) */
enum { SIM_BC_TRANSMISSIVE = 0, SIM_BC_PERIODIC = 1, SIM_BC_REFLECTIVE = 2, SIM_BC_INFLOW_FIXED = 3,
       SIM_BC_EXTERNAL = 4 /* x sides only: the two ghost columns belong to a neighbour slab (sim_slab_*) */ };
/* slope limiter ("van Leer non-smooth slope limiter"; R5): minmod form (default) or monotonised central */
enum { SIM_LIM_MINMOD = 0, SIM_LIM_MC = 1 };
/* field ids for sim_read_field */
enum { SIM_F_Q0 = 0, SIM_F_Q1, SIM_F_Q2, SIM_F_Q3, SIM_F_Q4, SIM_F_Q5, SIM_F_Q6,
       SIM_F_P = 16, SIM_F_T2 = 17, SIM_F_RHO = 18, SIM_F_U = 19, SIM_F_V = 20, SIM_F_LAMBDA = 21,
       SIM_F_PROGRESS = 22 /* 1 - lambda */, SIM_F_RHO2 = 23, SIM_F_C = 24, SIM_F_T1 = 25, SIM_F_RHO1 = 26 };
/* kernel variants (sim_set_variant): 0 = unfused reference kernels (halo, source, sweep, CFL as separate
   launches), 1 = fused production path (default). Both compute the same step. */
enum { SIM_VARIANT_UNFUSED = 0, SIM_VARIANT_FUSED = 1 };

typedef struct {
    int nx, ny;                 /* interior cells */
    double dx, dy;              /* metres */
    int bc_xlo, bc_xhi, bc_ylo, bc_yhi;
    double cfl;                 /* R11: dt = cfl * min(dx,dy) / max(max(|u|,|v|) + c) */
    int limiter;                /* SIM_LIM_* */
} sim_grid_t;

/* Table I, Table II, T_ref,2 = 0 K; z_min clamps the volume fractions */
typedef struct {
    double gamma1, cv1;
    double Gamma2, A, B, C, D, rho02, cv2, Tref2;
    double z_min;
} sim_eos_t;

/* Table III.  RK4 sub-stepping rule R13: n_sub = min(max_substeps, 1 + floor(theta/substep_theta)) */
typedef struct {
    double Ta, Cpre, Q;
    int reactive;               /* 0: inert (source step skipped); 1 needs Q, Cpre, Ta and eos cv2 > 0 (SIM_ERR_ARG otherwise) */
    int max_substeps;
    double substep_theta;
} sim_kin_t;

typedef struct { double x, y, r; } sim_cavity_t;   /* centre and radius in cell units */

/* problem setup.  Cavities come from exactly one of: explicit list (ncav > 0), square lattice
   (lattice != 0; Eq. 7 geometry), or the seeded generator (phi > 0; Eq. 8, R16). */
typedef struct {
    double p_shock;             /* input shock pressure [Pa]; slab i < shock_cells is set to the neat-NM Hugoniot state */
    int shock_cells;            /* L_s in cells */
    double p0, rho1_0, rho2_0;  /* ambient state */
    double interface_width;     /* tanh interface width in cells; h = width/2 (R15) */
    const sim_cavity_t* cav; int ncav;              /* HOST pointer, copied during the call */
    unsigned long long seed; double phi, dmin, dmax, min_gap; int x_lo, x_hi;
    int lattice; double lattice_d, lattice_spacing;
} sim_init_t;

typedef struct {
    double t; long long step; double dt_last, smax;
    double M2r, M2tot0, burned_mass, rate_inst;     /* Eq. 12-13 */
    double mass1, mass2, momx, momy, energy;        /* integrals of q0..q4 */
    int bad_state;
} sim_diag_t;

/* Bytes of device memory sim_create needs for this grid (0 on bad argument). Host-only computation. */
size_t sim_workspace_bytes(const sim_grid_t* grid);

/* Create a simulation. device_buf: DEVICE pointer to >= sim_workspace_bytes() bytes, 256-byte aligned, lent by
   the caller for the lifetime of the handle (e.g. a torch tensor), or NULL to let the library cudaMalloc it.
   cuda_stream: a cudaStream_t (NULL = default stream). [sync]
   If the driver cannot encode the tensor maps of the fused y-sweep (cuTensorMapEncodeTiled), the handle is still created, starts on
   SIM_VARIANT_UNFUSED, says so in sim_last_error(handle), and sim_set_variant(SIM_VARIANT_FUSED) returns SIM_ERR_CUDA. */
int sim_create(const sim_grid_t* grid, const sim_eos_t* eos, const sim_kin_t* kin,
               void* device_buf, size_t bytes, void* cuda_stream, sim_t** out);
void sim_destroy(sim_t*);
const char* sim_last_error(const sim_t*);          /* sim may be NULL: error of the last failed sim_create */

/* Initial condition on the device: cavity placement (generator R16 runs on the GPU), tanh painting,
   ambient state and shocked slab (O7).  Resets t, step; computes M2,tot and the first CFL dt. [sync] */
int sim_init(sim_t*, const sim_init_t*);
/* Explicit initial state from 7 HOST arrays of nx*ny doubles (row-major, x fastest).  q5 is clamped to
   [z_min, 1 - z_min] on entry (O3's clamp; a state the scheme produced is already inside and is stored unchanged). [sync] */
int sim_init_fields(sim_t*, const double* const host_q[7]);

/* CFL time step of the current state (a7). [sync] */
int sim_cfl_dt(sim_t*, double* dt_out);
/* n CFL-limited steps (O6: S(dt/2) X Y S(dt/2) on even steps, S Y X S on odd steps). [async] */
int sim_step(sim_t*, int n);
/* n steps with the given fixed dt (parity tests). [async] */
int sim_step_dt(sim_t*, int n, double dt);
/* Pieces of the step, exposed for parity tests: halo fill for a sweep direction (0 = x, 1 = y), one
   directional sweep (halo + MUSCL-Hancock/HLLC update), the source step over tau on every cell. [async] */
int sim_halo(sim_t*, int dir);
int sim_sweep(sim_t*, int dir, double dt);
int sim_source(sim_t*, double tau);

/* Global diagnostics (a8): Eq. 12 reactive mass, conservation integrals, instantaneous rate, S_max. [sync] */
int sim_diagnostics(sim_t*, sim_diag_t* out);
/* Copy one field (SIM_F_*) to host_out[nx*ny], row-major, x fastest. [sync] */
int sim_read_field(sim_t*, int field_id, double* host_out);
/* Cavity list used by the last sim_init (generator parity). Writes min(n, cap) entries. [sync] */
int sim_get_cavities(sim_t*, sim_cavity_t* host_out, int cap, int* n);
/* Seeded generator (R16; Eq. 8) of the last sim_init: the air fraction asked for and the one placed,
   pi sum r_k^2 / ((x_hi - x_lo) ny); both 0 when the layout was a list or a lattice.  sim_init returns SIM_ERR_ARG (and
   leaves the handle uninitialised) when the generator spends its candidate budget, 256 candidates per cavity of the
   target, before reaching the target: the list would silently describe another porosity.  These two numbers then say
   by how much. */
int sim_cavity_stats(const sim_t*, double* phi_target, double* phi_achieved);
/* Fused variant: how many warp segments the sweep kernels have repeated with the exact rules since the last sim_init*
   (a cell asked for RK4 sub-steps R13, for the first-order fallback R17, or held a liquid density outside the tables of
   the x^C, x^D evaluation).  0 on every run of the BASELINE configs; a large count means the fast
   path is being paid twice. [sync] */
int sim_redo_count(sim_t*, long long* n);

/* ---- post-processing of the state (the paper's analysis figures; R23-R26).  Not part of sim_step. ----
 * sim_profiles: y-averaged profiles Eq. 9-11 by the midpoint rule over the ny rows,
 *     pbar_i = (1/ny) sum_j p_ij,  rhobar_i = (1/ny) sum_j rho_ij,  ubar_i = sum_j (rho u)_ij / sum_j rho_ij,
 *   into HOST arrays of nx doubles (any of them may be NULL), and the leading-shock position of Appendix C,
 *     *xs_out = dx * (1 + max{i : pbar_i >= p_front})  [m], 0 if no column reaches p_front (the paper uses 1.01 p0).
 * sim_qdot_pdf: mass-weighted histogram of the volumetric energy-release rate, Eq. 14-16:
 *     qdot = q6 C exp(-Ta/T2) Q [W/m^3];  n = log10(qdot / 1e9);  b = floor((n - n_lo)/dn), counted iff 0 <= b < nbins;
 *     host_mass[b] += q1 dx dy  (mass of NM in the cell per unit depth),  host_count[b] += 1.
 *   Eq. 16's f = host_mass / (M2tot0 dn) is one division by the caller.  The paper's window is n_lo = 2, dn = 0.02,
 *   nbins = 400.  1 <= nbins <= 1024; either HOST output may be NULL.  An inert run returns zeros.
 * sim_shock_kinematics: Eq. C1-C2 on n HOST samples (host_t increasing, host_xs) with x_s(t) interpolated
 *   linearly: us_k = [x_s(t_k + dtau/2) - x_s(t_k - dtau/2)]/dtau, as_k = [x_s(t_k + dtau) - 2 x_s(t_k) + x_s(t_k - dtau)]/dtau^2,
 *   NaN where the window leaves [t_0, t_{n-1}].  n >= 2, dtau > 0 (the paper uses 1.5 us).
 * All three are [sync], deterministic (fixed summation shape) and allocate their scratch inside the library. */
int sim_profiles(sim_t*, double p_front, double* host_pbar, double* host_rhobar, double* host_ubar, double* xs_out);
int sim_qdot_pdf(sim_t*, double n_lo, double dn, int nbins, double* host_mass, long long* host_count);
int sim_shock_kinematics(sim_t*, const double* host_t, const double* host_xs, int n, double dtau, double* host_us, double* host_as);
/* sim_qdot_pdf for callers that must not touch the CUDA heap.  Same arguments, same kernels, same launch shape and
 * therefore bit-for-bit the same histogram as sim_qdot_pdf (Eq. 14-16), but the device scratch is a fixed
 * array inside libnmsdt.so's device image (about 2.3 MiB) instead of a buffer the handle grows with cudaMalloc.
 *   Meant for: (1) hosts that gave the whole GPU to their own arena and lend this library its workspace through
 *   sim_create's device_buf -- nothing is left for cudaMalloc to hand out, so sim_qdot_pdf fails there; (2) in-situ
 *   monitors that sample the histogram every few steps while other handles have sim_step work queued: cudaMalloc and
 *   cudaFree synchronise the whole device and would stall those queues at every sample.
 *   Limit: 1 <= nbins <= 512 (the paper's window has 400 bins); more returns SIM_ERR_ARG and sim_last_error names the
 *   limit.  The price: every GPU on which the library's kernels get loaded holds those 2.3 MiB until the process exits.
 *   This call, including its error paths, calls no cudaMalloc / cudaFree and no library routine that allocates device
 *   memory; host_mass / host_count are HOST arrays of nbins entries owned by the caller (either may be NULL) and are
 *   filled by plain device-to-host copies on the handle's stream.
 *   Set-up: the FIRST call on each device looks up the array's address on that device (cudaGetSymbolAddress) and raises
 *   the histogram kernel's shared-memory limit there; the device that holds the handle's state must be the current
 *   device (SIM_ERR_ARG otherwise).  Make that first call before starting any stream capture in the process.
 *   Sharing: there is ONE array per device, shared by all handles and all host threads, and it keeps the last call's
 *   contents (the call clears the part that has to start at zero itself).  Calls whose GPU work can overlap -- two
 *   handles on different streams of one device, from one thread or several -- race on it and return garbage; serialise
 *   them.  Calls on one handle are ordered by its stream and this call is [sync], so a single handle needs no care. */
int sim_qdot_pdf_noalloc(sim_t*, double n_lo, double dn, int nbins, double* host_mass, long long* host_count);

/* ---- multi-GPU slab decomposition along x (the paper names multi-GPU runs as future
 * work).  The domain is cut into slabs of whole columns, one handle (one GPU, one process) per slab.  A side
 * that faces another slab has the boundary kind SIM_BC_EXTERNAL: the halo step leaves its two ghost columns alone and
 * the caller fills them with the neighbour's two edge columns before every x-sweep (the only exchange of a step: the
 * y-sweep and the source step need nothing, stencil radius 2 in x, S8(e)); the time step needs the maximum wavespeed
 * over all slabs.  A step is driven piecewise (python: paper_1905_05727_b200/slab.py):
 *
 *     sim_slab_begin(s, dt_fixed)            local max wavespeed of the state -> the word sim_slab_smax_ptr points to
 *       <max-allreduce of that 8-byte word over the slabs>   (ordered bits of a non-negative double: integer max)
 *     sim_slab_ctl(s, 0)                     dt of the first step
 *     per step, for pass = 1, 2:
 *         if sim_slab_pass_dir(s, pass) == 0:  exchange: sim_slab_push (peer stores) or pack / transport / unpack
 *         sim_slab_pass(s, pass)             local halo + fused sweep (pass 2 leaves the new local max wavespeed)
 *       <max-allreduce>;  sim_slab_ctl(s, 1)   t += dt, step += 1, next dt
 *
 * Every slab then computes bit for bit what the single-handle run computes for its columns (same kernels, same dt).
 * All calls are [async] on the handle's stream unless marked; `pass` is 1 or 2, `side` is 0 (x-lo) or 1 (x-hi).
 * The exchanged block of one side is 7 planes x ny rows x 2 columns of doubles, dense in that order
 * (sim_slab_halo_bytes).  Fused variant only. */
typedef struct {
    void* plane0[2];            /* DEVICE pointers to plane 0 of the two plane sets (A: state between steps, B: between the passes) */
    long long plane_stride;     /* doubles between planes */
    int pitch, nx, ny;          /* doubles per row; interior size of that slab */
} sim_slab_peer_t;

/* sim_init for the slab whose first interior column is column x_origin of the global domain: `global_init` is the
   problem setup of the whole domain (shock_cells, cavity list / lattice / generator in global cell units; the seeded
   generator returns the same list on every slab), painted into this slab's columns. M2tot0 is the slab's share. [sync] */
int sim_init_slab(sim_t*, const sim_init_t* global_init, int x_origin);
size_t sim_slab_halo_bytes(const sim_t*);
int sim_slab_begin(sim_t*, double dt_fixed /* 0 = CFL-limited */);
int sim_slab_smax_ptr(sim_t*, void** device_word);          /* DEVICE pointer to the unsigned 64-bit max-wavespeed word */
int sim_slab_ctl(sim_t*, int advance);
int sim_slab_pass_dir(const sim_t*, int pass);             /* 0 = x, 1 = y for this pass of the current step; <0 on error */
int sim_slab_pass(sim_t*, int pass);
/* staging transport (NCCL send/recv, or any other): edge columns of this pass's input state -> dense DEVICE block,
   dense DEVICE block -> ghost columns of this pass's input state */
int sim_slab_pack(sim_t*, int pass, int side, void* device_out);
int sim_slab_unpack(sim_t*, int pass, int side, const void* device_in);
/* peer-store transport (NVLink / NVSwitch peer memory): describe this slab (sim_slab_info), hand a neighbour's
   description to sim_slab_connect (its pointers must be valid in this process: same process, or mapped through
   sim_slab_ipc_*), then sim_slab_push writes this slab's edge columns straight into the connected neighbours' ghost
   columns.  The caller orders push -> <barrier over the slabs> -> sim_slab_pass. peer = NULL disconnects. */
int sim_slab_info(const sim_t*, sim_slab_peer_t* out);
int sim_slab_connect(sim_t*, int side, const sim_slab_peer_t* peer);
int sim_slab_push(sim_t*, int pass);
/* CUDA IPC plumbing for the peer-store transport between processes: export the handle of this slab's workspace
   allocation (64 opaque bytes + the offsets of the two plane sets in it; needs a library-allocated workspace,
   device_buf = NULL in sim_create), open / close a neighbour's in this process. [sync] */
int sim_slab_ipc_export(const sim_t*, void* host_handle64, size_t* offset_A, size_t* offset_B);
int sim_slab_ipc_open(const void* host_handle64, void** device_base);
int sim_slab_ipc_close(void* device_base);

/* Select kernel variant (SIM_VARIANT_*) and whether sim_step replays CUDA graphs (default on). */
int sim_set_variant(sim_t*, int variant, int use_graph);
/* How sim_step enqueues the fused variant's kernels (2 per step: pass 1 and pass 2; ghost cells are taken from the
   boundary rule as the sweeps load them and the last block of pass 2 ends the step, so there is no halo or control
   launch): use_graph = pairs of steps replayed as one CUDA graph (default on), use_pdl = the kernels chained by
   programmatic dependent launch, a kernel's prologue overlapping its predecessor's tail (default off: on this two-launch
   step it measures equal on the smallest and the largest grids and 3 % slower on the 4096 x 512 one).  They change when
   kernels start, never what they compute. */
int sim_set_launch_mode(sim_t*, int use_graph, int use_pdl);
/* Launch geometry of the fused sweep in direction dir (0 = x, 1 = y) on this grid: a block (y: 256 columns, x: 4 rows)
   marches over *seg cells after *ramp recomputed ramp-up cells; *nblocks blocks per launch.  The kernels execute
   (seg + ramp)/seg times the algorithmic work: the roofline block of bench.py divides that out. */
int sim_sweep_geometry(const sim_t*, int dir, int* seg, int* ramp, long long* nblocks);
/* Number of kernel launches enqueued by this handle so far (bench.py's gpu_launches). */
long long sim_launch_count(const sim_t*);
/* Device pointer / layout of plane k of the current state (for zero-copy consumers). */
int sim_device_layout(const sim_t*, void** plane0, long long* plane_stride, int* pitch, int* x_offset, int* y_offset);
/* Per-kernel device timing with CUDA events on the handle's stream (bench.py's roofline block).
   sim_profile(s, 1) starts recording an event pair around every step kernel (graphs are bypassed while on);
   sim_profile(s, 0) stops and resolves them [sync]; sim_kernel_time returns the accumulated milliseconds and
   launch count of one kernel kind (SIM_K_*) since the last sim_profile(s, 1). */
enum { SIM_K_SWEEP_X = 0, SIM_K_SWEEP_Y = 1, SIM_K_SOURCE = 2, SIM_K_CFL = 3, SIM_K_HALO = 4, SIM_K_NKIND = 5 };
int sim_profile(sim_t*, int on);
int sim_kernel_time(const sim_t*, int kind, double* ms_total, long long* launches);
/* The measurement probes of bench.py and of the accuracy tests (sim_probe_fp64, sim_probe_issue, sim_probe_math) are not calls of
   the method: they are declared in include/nmsdt_probe.h. */

#ifdef __cplusplus
}
#endif
#endif
