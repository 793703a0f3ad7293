// nmsdt_capi.cu -- the C ABI of libnmsdt.so (include/nmsdt.h): handle, workspace layout, step orchestration.
#include "../../include/nmsdt.h"
#include "../../include/nmsdt_probe.h"
#include "nmsdt_host.h"
#include "nmsdt_math.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace nmsdt;

namespace {

std::string g_create_error;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
    int pitch, rows;
    long long fstride;       // doubles
    size_t off_A, off_B, off_inflow, off_partial, off_diag, off_diag0, off_ctl, off_scratch, off_tab, total;
};

Layout make_layout(int nx, int ny)
{
    Layout L;
    L.pitch = (int)align_up((size_t)(NGX + nx + NG), 16);
    L.rows = ny + 2 * NGY;
    L.fstride = (long long)L.pitch * L.rows;
    size_t plane_set = (size_t)7 * L.fstride * sizeof(double);
    size_t o = 0;
    L.off_A = o; o = align_up(o + plane_set, 256);
    L.off_B = o; o = align_up(o + plane_set, 256);
    L.off_inflow = o; o = align_up(o + (size_t)7 * ny * sizeof(double), 256);
    L.off_partial = o; o = align_up(o + (size_t)DIAG_BLOCKS * (DIAG_NV + 1) * sizeof(double), 256);
    L.off_diag = o; o = align_up(o + sizeof(DiagOut), 256);
    L.off_diag0 = o; o = align_up(o + sizeof(DiagOut), 256);
    L.off_ctl = o; o = align_up(o + sizeof(Ctl), 256);
    L.off_scratch = o; o = align_up(o + 8 * sizeof(double), 256);
    L.off_tab = o; o = align_up(o + MATH_TAB_DOUBLES_LOG * sizeof(double), 256);
    L.total = o;
    return L;
}

} // namespace

struct sim {
    sim_grid_t g;
    sim_eos_t e;
    sim_kin_t k;
    Params P;
    Layout L;
    cudaStream_t stream = nullptr;
    char* base = nullptr;
    bool owns = false;
    double *A = nullptr, *B = nullptr, *inflow = nullptr, *partial = nullptr, *scratch = nullptr, *tab = nullptr;
    DiagOut* d_diag = nullptr;
    Ctl* ctl = nullptr;
    Cav* d_cav = nullptr;
    int ncav = 0;
    double* post = nullptr;         // scratch of the post-processing calls (library-owned, grown on demand)
    size_t post_bytes = 0;
    bool inited = false;
    long long host_step = 0;        // mirrors ctl->step (step parity decides the sweep order)
    double M2tot0 = 0.0;
    bool m2tot0_pending = false;    // the reduction of the initial state is queued in d_diag0 and not read back yet
    DiagOut* d_diag0 = nullptr;
    double phi_target = 0.0, phi_achieved = 0.0;    // seeded generator: air fraction asked for / placed (0 without a generator)
    int variant = SIM_VARIANT_FUSED;
    int use_graph = 1;
    int use_pdl = 0;                // chain the kernels of sim_step by programmatic dependent launch (measured slower: off)
    cudaGraphExec_t gexec = nullptr;    // fused path: one even (X-Y) + one odd (Y-X) step = 4 kernel nodes
    cudaStream_t cap_stream = nullptr;  // private stream the graph is captured on (the caller's may be the legacy stream)
    bool graph_failed = false;
    bool cfl_valid = false;         // fused path: ctl->dt / ctl->tsafe describe the current state and dt mode
    double dt_mode = -1.0;          // dt_fixed the control block was last prepared for
    long long launches = 0;
    std::string err;
    bool tm_ok = true;              // false: the tensor maps could not be encoded, the handle is confined to the unfused variant
    CUtensorMap tmA, tmB;           // the two plane sets as {pitch, rows, 7} tensors with a {32, 1, 7} box (y-sweep staging)
    sim_slab_peer_t peer[2];        // slab decomposition: connected neighbours (peer-store transport)
    bool peer_on[2] = {false, false};
    // event profiling (sim_profile)
    struct EvPair { cudaEvent_t a, b; int kind; };
    std::vector<EvPair> ev;
    size_t ev_used = 0;
    bool profile = false;
    double kms[SIM_K_NKIND] = {0, 0, 0, 0, 0};
    long long kcount[SIM_K_NKIND] = {0, 0, 0, 0, 0};
};

namespace {

int fail(sim* s, int code, const std::string& msg)
{
    if (s) s->err = msg; else g_create_error = msg;
    return code;
}

int check_cuda(sim* s, const char* what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(s, SIM_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
    return SIM_OK;
}

bool grid_ok(const sim_grid_t* g)
{
    if (!g || g->nx < 1 || g->ny < 1 || !(g->dx > 0.0) || !(g->dy > 0.0) || !(g->cfl > 0.0)) return false;
    const int b[4] = {g->bc_xlo, g->bc_xhi, g->bc_ylo, g->bc_yhi};
    for (int i = 0; i < 4; ++i) if (b[i] < 0 || b[i] > (i < 2 ? SIM_BC_EXTERNAL : 3)) return false;
    if (g->bc_xhi == SIM_BC_INFLOW_FIXED || g->bc_ylo == SIM_BC_INFLOW_FIXED || g->bc_yhi == SIM_BC_INFLOW_FIXED) return false;
    if ((g->bc_xlo == SIM_BC_PERIODIC) != (g->bc_xhi == SIM_BC_PERIODIC)) return false;
    if ((g->bc_ylo == SIM_BC_PERIODIC) != (g->bc_yhi == SIM_BC_PERIODIC)) return false;
    if (g->limiter != SIM_LIM_MINMOD && g->limiter != SIM_LIM_MC) return false;
    return true;
}

void fill_params(sim* s)
{
    Params& P = s->P;
    const sim_grid_t& g = s->g; const sim_eos_t& e = s->e; const sim_kin_t& k = s->k;
    P.nx = g.nx; P.ny = g.ny; P.pitch = s->L.pitch; P.rows = s->L.rows; P.fstride = s->L.fstride;
    P.dx = g.dx; P.dy = g.dy; P.cfl = g.cfl; P.hmin = g.dx < g.dy ? g.dx : g.dy;
    P.bc_xlo = g.bc_xlo; P.bc_xhi = g.bc_xhi; P.bc_ylo = g.bc_ylo; P.bc_yhi = g.bc_yhi; P.limiter = g.limiter;
    P.gamma1 = e.gamma1; P.G1 = e.gamma1 - 1.0; P.iG1 = 1.0 / P.G1; P.cv1 = e.cv1;
    P.G2 = e.Gamma2; P.iG2 = 1.0 / e.Gamma2; P.G2p1 = e.Gamma2 + 1.0;
    P.A = e.A; P.B = e.B; P.C = e.C; P.D = e.D; P.rho02 = e.rho02; P.irho02 = 1.0 / e.rho02; P.cv2 = e.cv2; P.Tref2 = e.Tref2;
    P.kA = -e.A / (1.0 - e.C); P.kB = e.B / (1.0 - e.D); P.AC = e.A * e.C; P.BD = e.B * e.D;
    P.z_min = e.z_min; P.z_max = 1.0 - e.z_min;
    P.C2 = e.C * LOG2E; P.D2 = e.D * LOG2E; P.iG2cv2 = 1.0 / (e.Gamma2 * e.cv2); P.tab = s->tab; P.inflow = s->inflow;
    fill_pow_coef(P.pw, e.C, e.D);
    P.g1iG1 = e.gamma1 / (e.gamma1 - 1.0);
    // rho2 e_ref2 - p_ref2/Gamma2 = E1 x^C + E2 x^D - E3 x and rho2 c2^2 - (Gamma2+1) p = R1 x^C + R2 x^D  (Eq. 3-4 in O2)
    P.E1 = P.kA - e.A / e.Gamma2; P.E2 = P.kB + e.B / e.Gamma2; P.E3 = P.kA + P.kB;
    P.R1 = e.A * (e.C - (e.Gamma2 + 1.0)); P.R2 = e.B * ((e.Gamma2 + 1.0) - e.D);
    P.Ta = k.Ta; P.Cpre = k.Cpre; P.Q = k.Q; P.theta0 = k.substep_theta; P.reactive = k.reactive; P.max_substeps = k.max_substeps;
}

// Shocked-slab state (O7): the neat-liquid Hugoniot point at pressure ps, found in the specific volume v = 1/rho.
// With Eq. 2 solved for e (constant Gamma2) the Hugoniot condition e - e0 = (ps + p0)(v0 - v)/2 reads
//     h(v) = e_ref(v) + v (ps - p_ref(v))/Gamma2 - e0 - (ps + p0)(v0 - v)/2 = 0,
// and since Eq. 3-4 satisfy de_ref/dv = -p_ref,
//     h'(v) = -p_ref + (ps - p_ref)/Gamma2 - v p_ref'(v)/Gamma2 + (ps + p0)/2,   v p_ref'(v) = -(A C x^C - B D x^D),  x = 1/(rho02 v).
// Newton from v0, kept inside a bracket that every iterate tightens (h(v0) > 0 for ps > p0; h < 0 towards the compression
// limit v0 Gamma2/(Gamma2 + 2)); written apart from the oracle's bisection in rho.
struct HugFn {
    const sim_eos_t& e; double ps, p0, v0, e0;
    static void ref(const sim_eos_t& e, double v, double& pr, double& er, double& vdpr)
    {
        const double x = 1.0 / (e.rho02 * v), xC = std::pow(x, e.C), xD = std::pow(x, e.D);
        pr = e.A * xC - e.B * xD;                                                              // Eq. 3
        er = (-e.A / (1.0 - e.C) * (xC / x - 1.0) + e.B / (1.0 - e.D) * (xD / x - 1.0)) / e.rho02;   // Eq. 4
        vdpr = -(e.A * e.C * xC - e.B * e.D * xD);
    }
    void eval(double v, double& h, double& dh) const
    {
        double pr, er, vdpr;
        ref(e, v, pr, er, vdpr);
        h = er + v * (ps - pr) / e.Gamma2 - e0 - 0.5 * (ps + p0) * (v0 - v);
        dh = -pr + (ps - pr) / e.Gamma2 - vdpr / e.Gamma2 + 0.5 * (ps + p0);
    }
};

bool hugoniot(const sim_eos_t& e, double p0, double rho1_0, double rho2_0, double ps, Hug& out)
{
    if (!(ps > p0) || !(rho2_0 > 0.0)) return false;
    const double v0 = 1.0 / rho2_0;
    double pr0, er0, t0;
    HugFn::ref(e, v0, pr0, er0, t0);
    const HugFn F{e, ps, p0, v0, er0 + v0 * (p0 - pr0) / e.Gamma2};
    double hi = v0, lo = v0 * e.Gamma2 / (e.Gamma2 + 2.0) * 0.5, h, dh;
    F.eval(lo, h, dh);
    for (int it = 0; it < 60 && !(h < 0.0); ++it) { lo *= 0.5; F.eval(lo, h, dh); }
    if (!(h < 0.0)) return false;
    double v = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        F.eval(v, h, dh);
        if (h > 0.0) hi = v; else lo = v;
        double vn = v - h / dh;
        if (!(vn > lo && vn < hi)) vn = 0.5 * (lo + hi);            // safeguard: bisect when Newton leaves the bracket
        if (std::fabs(vn - v) <= 1e-16 * v) { v = vn; break; }
        v = vn;
    }
    const double rs = 1.0 / v;
    double prs, ers, ts;
    HugFn::ref(e, v, prs, ers, ts);
    out.rho_s = rs;
    out.u_p = std::sqrt((ps - p0) * (v0 - v));
    out.U_s = v0 * std::sqrt((ps - p0) / (v0 - v));                 // mass + momentum jump: (rho0 U_s)^2 = (ps - p0)/(v0 - v)
    out.T2_s = e.Tref2 + (ps - prs) * v / (e.Gamma2 * e.cv2);       // Eq. 5
    const double g = e.gamma1;
    out.rho1_s = rho1_0 * ((g + 1.0) * ps + (g - 1.0) * p0) / ((g - 1.0) * ps + (g + 1.0) * p0);    // trace air: its own shock Hugoniot
    return true;
}

// Tensor map of one plane set for the y-sweep's bulk row copies: fp64 tensor {pitch, rows, 7 planes} (x fastest), box
// {32 columns, 1 row, 7 planes}, no swizzle, out-of-range columns read as zero.  The encoder lives in the driver library;
// it is fetched through the runtime so that libnmsdt.so links against nothing but libcudart.
bool make_plane_tensor_map(CUtensorMap* tm, const double* plane0, int pitch, int rows, long long fstride)
{
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;
    static std::once_flag once;                      // handles may be created from several host threads at once
    std::call_once(once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess && fn) encode = (encode_fn)fn;
        else cudaGetLastError();
    });
    if (!encode) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)pitch, (cuuint64_t)rows, 7};
    const cuuint64_t strides[2] = {(cuuint64_t)pitch * sizeof(double), (cuuint64_t)fstride * sizeof(double)};     // bytes, dims 1 and 2
    const cuuint32_t box[3] = {32, 1, 7}, estr[3] = {1, 1, 1};
    return encode(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)plane0, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// event pair around one kernel launch while profiling
struct KTimer {
    sim* s; int idx = -1;
    KTimer(sim* s_, int kind) : s(s_)
    {
        if (!s->profile) return;
        if (s->ev_used == s->ev.size()) {
            sim::EvPair p; cudaEventCreate(&p.a); cudaEventCreate(&p.b); p.kind = kind;
            s->ev.push_back(p);
        }
        idx = (int)s->ev_used++;
        s->ev[idx].kind = kind;
        cudaEventRecord(s->ev[idx].a, s->stream);
    }
    ~KTimer() { if (idx >= 0) cudaEventRecord(s->ev[idx].b, s->stream); }
};

// one full step on the unfused reference path: CFL, S(dt/2), sweep, sweep, S(dt/2)
void enqueue_step_unfused(sim* s)
{
    cudaStream_t st = s->stream;
    const Params& P = s->P;
    { KTimer t(s, SIM_K_CFL); launch_cfl(P, s->A, s->ctl, st); }
    launch_finalize_dt(P, s->ctl, st);
    s->launches += 2;
    const double* dtp = &s->ctl->dt;
    if (P.reactive) { KTimer t(s, SIM_K_SOURCE); launch_source(P, s->A, dtp, 0.5, st); s->launches++; }
    const int d1 = (s->host_step & 1) ? 1 : 0, d2 = 1 - d1;
    { KTimer t(s, SIM_K_HALO); launch_halo(P, s->A, s->inflow, d1, st); }
    { KTimer t(s, d1 == 0 ? SIM_K_SWEEP_X : SIM_K_SWEEP_Y); launch_sweep_march(P, s->A, s->B, dtp, d1, st); }
    { KTimer t(s, SIM_K_HALO); launch_halo(P, s->B, s->inflow, d2, st); }
    { KTimer t(s, d2 == 0 ? SIM_K_SWEEP_X : SIM_K_SWEEP_Y); launch_sweep_march(P, s->B, s->A, dtp, d2, st); }
    s->launches += 4;
    if (P.reactive) { KTimer t(s, SIM_K_SOURCE); launch_source(P, s->A, dtp, 0.5, st); s->launches++; }
    launch_advance(s->ctl, st);
    s->launches++;
    s->host_step++;
}

// one full step on the fused path: [S(dt/2) + sweep d1] [sweep d2 + S(dt/2) + CFL partial + end of step]
void enqueue_step_fused(sim* s)
{
    cudaStream_t st = s->stream;
    const Params& P = s->P;
    const double* dtp = &s->ctl->dt;
    const int d1 = (s->host_step & 1) ? 1 : 0, d2 = 1 - d1;
    const bool pdl = s->use_pdl && !s->profile;      // (event pairs between the kernels would serialise them anyway)
    // (no halo launches: the fused sweeps take ghost cells from the boundary rule as they load them, ghost_src in nmsdt_fused.cu)
    { KTimer t(s, d1 == 0 ? SIM_K_SWEEP_X : SIM_K_SWEEP_Y); launch_sweep_fused(P, s->A, &s->tmA, s->B, dtp, s->ctl, d1, 1, st, pdl); }
    // (the step is ended -- t, step counter, next dt -- by the last block of the pass-2 sweep to finish: no k_ctl launch)
    { KTimer t(s, d2 == 0 ? SIM_K_SWEEP_X : SIM_K_SWEEP_Y); launch_sweep_fused(P, s->B, &s->tmB, s->A, dtp, s->ctl, d2, 2, st, pdl, true); }
    s->launches += 2;
    s->host_step++;
}

// fused path: CUDA graph of two consecutive steps (2 x 2 kernels) starting at an even step.  Captured once on a private stream
// (nothing executes during capture; every kernel argument is fixed for the lifetime of the handle) and replayed on
// the caller's stream, which removes the per-launch CPU cost that dominates the small configs (C1, C2).
bool ensure_graph(sim* s)
{
    if (s->gexec) return true;
    if (s->graph_failed) return false;
    s->graph_failed = true;
    if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return false; }
    cudaStream_t user = s->stream;
    const long long step0 = s->host_step, l0 = s->launches;
    cudaGraph_t g = nullptr;
    if (cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return false; }
    s->stream = s->cap_stream;
    s->host_step = 0;
    enqueue_step_fused(s);
    enqueue_step_fused(s);
    s->stream = user; s->host_step = step0; s->launches = l0;
    if (cudaStreamEndCapture(s->cap_stream, &g) != cudaSuccess || !g) { cudaGetLastError(); return false; }
    const cudaError_t e = cudaGraphInstantiate(&s->gexec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { cudaGetLastError(); s->gexec = nullptr; return false; }
    s->graph_failed = false;
    return true;
}

// fused path: make ctl->dt / ctl->tsafe valid for the current state (first step after init or after a piecewise call)
void prepare_ctl_fused(sim* s)
{
    { KTimer t(s, SIM_K_CFL); launch_cfl(s->P, s->A, s->ctl, s->stream); }
    launch_ctl(s->P, s->ctl, 0, s->stream);
    s->launches += 2;
}

// End of sim_init / sim_init_fields: inflow column, control block and the reduction of the initial state (M2tot0 of
// Eq. 13 is M2r at t = 0) are queued behind the caller's data; the one synchronisation that follows also ends the
// library's use of the caller's host buffers.  The reduced sums stay on the device until the first sim_diagnostics.
int finish_init(sim* s)
{
    cudaStream_t st = s->stream;
    launch_capture_inflow(s->P, s->A, s->inflow, st);
    cudaMemsetAsync(s->ctl, 0, sizeof(Ctl), st);
    launch_diag(s->P, s->A, s->partial, s->d_diag0, st);
    s->launches += 3;
    s->host_step = 0;
    s->cfl_valid = false;
    s->M2tot0 = 0.0;
    s->m2tot0_pending = true;
    if (cudaStreamSynchronize(st) != cudaSuccess) return check_cuda(s, "init");
    s->inited = true;
    return check_cuda(s, "init");
}

} // namespace

extern "C" {

size_t sim_workspace_bytes(const sim_grid_t* g)
{
    if (!grid_ok(g)) return 0;
    return make_layout(g->nx, g->ny).total;
}

const char* sim_last_error(const sim_t* s) { return s ? s->err.c_str() : g_create_error.c_str(); }

int sim_create(const sim_grid_t* g, const sim_eos_t* e, const sim_kin_t* k, void* device_buf, size_t bytes, void* cuda_stream, sim_t** out)
{
    if (!out) return fail(nullptr, SIM_ERR_ARG, "sim_create: out is NULL");
    *out = nullptr;
    if (!grid_ok(g) || !e || !k) return fail(nullptr, SIM_ERR_ARG, "sim_create: bad grid / eos / kin argument");
    if (!(e->z_min > 0.0 && e->z_min < 0.5) || !(e->gamma1 > 1.0) || !(e->Gamma2 > 0.0) || !(e->rho02 > 0.0) || e->C == 1.0 || e->D == 1.0)
        return fail(nullptr, SIM_ERR_ARG, "sim_create: bad EOS parameters");
    if (k->max_substeps < 1 || !(k->substep_theta > 0.0)) return fail(nullptr, SIM_ERR_ARG, "sim_create: bad kinetics parameters");
    // the fused source step decides all four RK4 stages by one T2 > 0 test (rk4_step, nmsdt_fast.cuh): that is the oracle's per-stage
    // test only for an exothermic, forward reaction (beta = Q/cv2 > 0, C > 0, Ta > 0; Table II-III), so nothing else is taken
    if (k->reactive && (!(k->Q > 0.0) || !(e->cv2 > 0.0) || !(k->Cpre > 0.0) || !(k->Ta > 0.0)))
        return fail(nullptr, SIM_ERR_ARG, "sim_create: a reactive run needs Q > 0, cv2 > 0, Cpre > 0 and Ta > 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, SIM_ERR_CUDA, "sim_create: no CUDA device (libnmsdt has no CPU fallback)");
    }
    sim* s = new sim();
    s->g = *g; s->e = *e; s->k = *k;
    s->L = make_layout(g->nx, g->ny);
    if (s->L.fstride >= (1LL << 32)) { delete s; return fail(nullptr, SIM_ERR_ARG, "sim_create: a plane of 2^32 doubles or more (34 GB) is not supported"); }
    s->stream = (cudaStream_t)cuda_stream;
    if (device_buf) {
        if (bytes < s->L.total || ((uintptr_t)device_buf & 255)) { delete s; return fail(nullptr, SIM_ERR_ARG, "sim_create: device_buf too small or not 256-byte aligned"); }
        s->base = (char*)device_buf;
    } else {
        if (cudaMalloc(&s->base, s->L.total) != cudaSuccess) { cudaGetLastError(); delete s; return fail(nullptr, SIM_ERR_CUDA, "sim_create: cudaMalloc failed"); }
        s->owns = true;
    }
    s->A = (double*)(s->base + s->L.off_A); s->B = (double*)(s->base + s->L.off_B);
    s->inflow = (double*)(s->base + s->L.off_inflow); s->partial = (double*)(s->base + s->L.off_partial);
    s->d_diag = (DiagOut*)(s->base + s->L.off_diag); s->d_diag0 = (DiagOut*)(s->base + s->L.off_diag0); s->ctl = (Ctl*)(s->base + s->L.off_ctl);
    s->scratch = (double*)(s->base + s->L.off_scratch);
    s->tab = (double*)(s->base + s->L.off_tab);
    fill_params(s);
    if (!make_plane_tensor_map(&s->tmA, s->A, s->L.pitch, s->L.rows, s->L.fstride) || !make_plane_tensor_map(&s->tmB, s->B, s->L.pitch, s->L.rows, s->L.fstride)) {
        // only the fused y-sweep stages its rows with bulk tensor copies: the unfused kernels, the x-only piecewise calls, diagnostics
        // and post-processing do without.  The handle starts on the unfused variant and sim_set_variant refuses the fused one.
        s->tm_ok = false;
        s->variant = SIM_VARIANT_UNFUSED;
        s->err = "sim_create: cuTensorMapEncodeTiled is unavailable or failed; this handle runs SIM_VARIANT_UNFUSED only";
    }
    init_fused_kernels();
    cudaMemsetAsync(s->base, 0, s->L.total, s->stream);
    {
        double htab[MATH_TAB_DOUBLES_LOG];
        fill_math_tables(htab, e->C, e->D);
        cudaMemcpyAsync(s->tab, htab, sizeof(htab), cudaMemcpyHostToDevice, s->stream);   // pageable source: staged before return
    }
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) { int rc = check_cuda(nullptr, "sim_create"); sim_destroy(s); return rc ? rc : SIM_ERR_CUDA; }
    *out = s;
    return SIM_OK;
}

void sim_destroy(sim_t* s)
{
    if (!s) return;
    cudaStreamSynchronize(s->stream);
    if (s->d_cav) cudaFree(s->d_cav);
    if (s->post) cudaFree(s->post);
    if (s->gexec) cudaGraphExecDestroy(s->gexec);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    for (auto& p : s->ev) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    if (s->owns && s->base) cudaFree(s->base);
    delete s;
}

// sim_init of the slab whose first interior column is global column x0 (x0 = 0, whole domain: sim_init)
static int init_common(sim_t* s, const sim_init_t* in, int x0, bool slab)
{
    if (!s || !in) return fail(s, SIM_ERR_ARG, "sim_init: NULL argument");
    if (in->shock_cells < 0 || (!slab && in->shock_cells > s->g.nx) || !(in->interface_width > 0.0)) return fail(s, SIM_ERR_ARG, "sim_init: bad shock_cells / interface_width");
    cudaStream_t st = s->stream;
    const Params& P = s->P;
    s->inited = false;              // until finish_init: a failed sim_init leaves no half-written state behind a valid handle
    if (s->d_cav) { cudaFree(s->d_cav); s->d_cav = nullptr; }
    s->ncav = 0; s->phi_target = s->phi_achieved = 0.0;
    std::vector<Cav> host;
    if (in->cav && in->ncav > 0) {
        for (int i = 0; i < in->ncav; ++i) host.push_back({in->cav[i].x - x0, in->cav[i].y, in->cav[i].r});
    } else if (in->lattice) {     // R20: centres x_lo + s/2 + s i, s/2 + s j
        if (!(in->lattice_spacing > 0.0) || !(in->lattice_d > 0.0)) return fail(s, SIM_ERR_ARG, "sim_init: bad lattice");
        const double sp = in->lattice_spacing, r = 0.5 * in->lattice_d;
        for (int jj = 0; sp * (jj + 1) <= (double)s->g.ny; ++jj)
            for (int ii = 0; in->x_lo + sp * (ii + 1) <= (double)in->x_hi; ++ii) host.push_back({in->x_lo + 0.5 * sp + sp * ii - x0, 0.5 * sp + sp * jj, r});
    } else if (in->phi > 0.0) {
        long long sum_r2 = 0, target_r2 = 0;
        int n = generate_cavities(in->seed, in->phi, in->dmin, in->dmax, in->min_gap, in->x_lo, in->x_hi, s->g.ny,
                                  s->g.bc_ylo == SIM_BC_PERIODIC ? 1 : 0, &s->d_cav, st, &s->launches, &sum_r2, &target_r2);
        if (n == -1) return fail(s, SIM_ERR_ARG, "sim_init: bad generator parameters");
        if (n < 0) { cudaGetLastError(); return fail(s, SIM_ERR_CUDA, "sim_init: cavity generator failed"); }
        s->ncav = n;
        // air fraction placed: pi sum r^2 over the seeded region (r in 1/256 cell)
        const double region = (double)(in->x_hi - in->x_lo) * (double)s->g.ny * 65536.0 / 3.14159265358979323846;
        s->phi_target = in->phi; s->phi_achieved = (double)sum_r2 / region;
        if (sum_r2 < target_r2) {
            char msg[256];
            std::snprintf(msg, sizeof msg, "sim_init: the seeded generator placed %d cavities = air fraction %.5f of the %.5f asked for "
                          "(candidate budget spent: the target is at or beyond the jamming limit of this minimum gap)", n, s->phi_achieved, in->phi);
            return fail(s, SIM_ERR_ARG, msg);
        }
        if (x0 != 0 && n > 0) { launch_shift_cavities(s->d_cav, n, -(double)x0, st); s->launches++; }
    }
    if (!host.empty()) {
        if (cudaMalloc(&s->d_cav, sizeof(Cav) * host.size()) != cudaSuccess) { cudaGetLastError(); return fail(s, SIM_ERR_CUDA, "sim_init: cudaMalloc"); }
        cudaMemcpyAsync(s->d_cav, host.data(), sizeof(Cav) * host.size(), cudaMemcpyHostToDevice, st);
        cudaStreamSynchronize(st);
        s->ncav = (int)host.size();
    }
    Hug hug = {0, 0, 0, 0, 0};
    if (in->shock_cells > 0 && !hugoniot(s->e, in->p0, in->rho1_0, in->rho2_0, in->p_shock, hug)) return fail(s, SIM_ERR_ARG, "sim_init: Hugoniot solve failed");
    launch_zero_plane(P, s->A + 5 * P.fstride, st);
    launch_paint(P, s->A + 5 * P.fstride, s->d_cav, s->ncav, 0.5 * in->interface_width, st);
    const int sc_local = in->shock_cells - x0 < 0 ? 0 : (in->shock_cells - x0 > s->g.nx ? s->g.nx : in->shock_cells - x0);
    launch_fill_state(P, s->A, sc_local, hug, in->p_shock, in->p0, in->rho1_0, in->rho2_0, st);
    s->launches += 3;
    return finish_init(s);
}

int sim_init(sim_t* s, const sim_init_t* in) { return init_common(s, in, 0, false); }
int sim_init_slab(sim_t* s, const sim_init_t* in, int x_origin) { return init_common(s, in, x_origin, true); }

int sim_init_fields(sim_t* s, const double* const host_q[7])
{
    if (!s || !host_q) return fail(s, SIM_ERR_ARG, "sim_init_fields: NULL argument");
    const Params& P = s->P;
    for (int f = 0; f < 7; ++f) {
        if (!host_q[f]) return fail(s, SIM_ERR_ARG, "sim_init_fields: NULL plane");
        double* dst = s->A + f * P.fstride + (long long)NGY * P.pitch + NGX;
        if (cudaMemcpy2DAsync(dst, (size_t)P.pitch * 8, host_q[f], (size_t)P.nx * 8, (size_t)P.nx * 8, P.ny, cudaMemcpyHostToDevice, s->stream) != cudaSuccess)
            return check_cuda(s, "sim_init_fields");
    }
    launch_clamp_z1(P, s->A + 5 * P.fstride, s->stream);       // q5 within [z_min, 1 - z_min]: the invariant of every stored state
    s->launches++;
    const int rc = finish_init(s);                              // (synchronises: the host planes are free again)
    if (s->d_cav) { cudaFree(s->d_cav); s->d_cav = nullptr; }
    s->ncav = 0; s->phi_target = s->phi_achieved = 0.0;
    return rc;
}

int sim_cfl_dt(sim_t* s, double* dt_out)
{
    if (!s || !dt_out) return fail(s, SIM_ERR_ARG, "sim_cfl_dt: NULL argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_cfl_dt: not initialised");
    s->cfl_valid = false;
    launch_set_double(&s->ctl->dt_fixed, 0.0, s->stream);
    launch_cfl(s->P, s->A, s->ctl, s->stream);
    launch_finalize_dt(s->P, s->ctl, s->stream);
    s->launches += 3;
    Ctl h;
    cudaMemcpyAsync(&h, s->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_cfl_dt");
    *dt_out = h.dt;
    if (h.bad) return fail(s, SIM_ERR_BAD, "sim_cfl_dt: non-finite or non-positive state");
    return SIM_OK;
}

static int step_common(sim_t* s, int n, double dt_fixed)
{
    if (!s || n < 0) return fail(s, SIM_ERR_ARG, "sim_step: bad argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_step: not initialised");
    launch_set_double(&s->ctl->dt_fixed, dt_fixed, s->stream);
    s->launches++;
    if (s->variant == SIM_VARIANT_UNFUSED) {
        for (int it = 0; it < n; ++it) enqueue_step_unfused(s);
        s->cfl_valid = false;
        return check_cuda(s, "sim_step");
    }
    if (n == 0) return SIM_OK;
    if (!s->cfl_valid || s->dt_mode != dt_fixed) prepare_ctl_fused(s);
    if (s->use_graph && !s->profile && n >= 3) {
        if (s->host_step & 1) { enqueue_step_fused(s); --n; }
        if (ensure_graph(s)) {
            for (; n >= 2; n -= 2) {
                if (cudaGraphLaunch(s->gexec, s->stream) != cudaSuccess) return check_cuda(s, "sim_step (graph)");
                s->launches += 4; s->host_step += 2;
            }
        }
    }
    for (int it = 0; it < n; ++it) enqueue_step_fused(s);
    s->cfl_valid = true; s->dt_mode = dt_fixed;
    return check_cuda(s, "sim_step");
}

int sim_step(sim_t* s, int n) { return step_common(s, n, 0.0); }

int sim_step_dt(sim_t* s, int n, double dt)
{
    if (!(dt > 0.0)) return fail(s, SIM_ERR_ARG, "sim_step_dt: dt must be positive");
    return step_common(s, n, dt);
}

int sim_halo(sim_t* s, int dir)
{
    if (!s || (dir != 0 && dir != 1)) return fail(s, SIM_ERR_ARG, "sim_halo: bad argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_halo: not initialised");
    launch_halo(s->P, s->A, s->inflow, dir, s->stream);
    s->launches++;
    return check_cuda(s, "sim_halo");
}

int sim_sweep(sim_t* s, int dir, double dt)
{
    if (!s || (dir != 0 && dir != 1) || !(dt > 0.0)) return fail(s, SIM_ERR_ARG, "sim_sweep: bad argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_sweep: not initialised");
    s->cfl_valid = false;
    launch_set_double(s->scratch, dt, s->stream);
    launch_set_double(s->scratch + 1, 1e300, s->stream);
    launch_halo(s->P, s->A, s->inflow, dir, s->stream);
    if (s->variant == SIM_VARIANT_FUSED) launch_sweep_fused(s->P, s->A, &s->tmA, s->B, s->scratch, s->ctl, dir, 0, s->stream);
    else launch_sweep_march(s->P, s->A, s->B, s->scratch, dir, s->stream);
    s->launches += 4;
    // keep the state in A: copy the interior planes back (parity-test helper, not on the hot path)
    cudaMemcpyAsync(s->A, s->B, (size_t)7 * s->P.fstride * sizeof(double), cudaMemcpyDeviceToDevice, s->stream);
    return check_cuda(s, "sim_sweep");
}

int sim_source(sim_t* s, double tau)
{
    if (!s || !(tau > 0.0)) return fail(s, SIM_ERR_ARG, "sim_source: bad argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_source: not initialised");
    if (!s->P.reactive) return SIM_OK;
    s->cfl_valid = false;
    launch_set_double(s->scratch, tau, s->stream);
    if (s->variant == SIM_VARIANT_FUSED) {
        launch_set_double(s->scratch + 1, host_tsafe(tau, s->k.Cpre, s->k.Ta, s->k.substep_theta), s->stream);
        launch_source_fast(s->P, s->A, s->scratch, s->stream);
        s->launches++;
    } else launch_source(s->P, s->A, s->scratch, 1.0, s->stream);
    s->launches += 2;
    return check_cuda(s, "sim_source");
}

int sim_diagnostics(sim_t* s, sim_diag_t* out)
{
    if (!s || !out) return fail(s, SIM_ERR_ARG, "sim_diagnostics: NULL argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_diagnostics: not initialised");
    launch_diag(s->P, s->A, s->partial, s->d_diag, s->stream);
    s->launches += 2;
    DiagOut d, d0; Ctl c;
    if (s->m2tot0_pending) cudaMemcpyAsync(&d0, s->d_diag0, sizeof(DiagOut), cudaMemcpyDeviceToHost, s->stream);
    cudaMemcpyAsync(&d, s->d_diag, sizeof(DiagOut), cudaMemcpyDeviceToHost, s->stream);
    cudaMemcpyAsync(&c, s->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_diagnostics");
    const double dA = s->g.dx * s->g.dy;
    if (s->m2tot0_pending) { s->M2tot0 = d0.sum[5] * dA; s->m2tot0_pending = false; }
    out->t = c.t; out->step = c.step; out->dt_last = c.dt_last; out->smax = d.smax;
    out->M2r = d.sum[5] * dA; out->M2tot0 = s->M2tot0; out->burned_mass = s->M2tot0 - out->M2r; out->rate_inst = d.sum[6] * dA;
    out->mass1 = d.sum[0] * dA; out->mass2 = d.sum[1] * dA; out->momx = d.sum[2] * dA; out->momy = d.sum[3] * dA; out->energy = d.sum[4] * dA;
    out->bad_state = (d.bad || c.bad) ? 1 : 0;
    if (out->bad_state) return fail(s, SIM_ERR_BAD, "sim_diagnostics: non-finite or non-positive state");
    return check_cuda(s, "sim_diagnostics");
}

int sim_read_field(sim_t* s, int fid, double* host_out)
{
    if (!s || !host_out) return fail(s, SIM_ERR_ARG, "sim_read_field: NULL argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_read_field: not initialised");
    const Params& P = s->P;
    if (fid >= 0 && fid < 7) {
        const double* src = s->A + fid * P.fstride + (long long)NGY * P.pitch + NGX;
        cudaMemcpy2DAsync(host_out, (size_t)P.nx * 8, src, (size_t)P.pitch * 8, (size_t)P.nx * 8, P.ny, cudaMemcpyDeviceToHost, s->stream);
    } else if (fid >= 16 && fid <= 26) {
        double* dense = s->B;    // B is free between steps
        launch_derived(P, s->A, fid, dense, s->stream);
        s->launches++;
        cudaMemcpyAsync(host_out, dense, (size_t)P.nx * P.ny * 8, cudaMemcpyDeviceToHost, s->stream);
    } else return fail(s, SIM_ERR_ARG, "sim_read_field: unknown field id");
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_read_field");
    return check_cuda(s, "sim_read_field");
}

int sim_get_cavities(sim_t* s, sim_cavity_t* host_out, int cap, int* n)
{
    if (!s || !n) return fail(s, SIM_ERR_ARG, "sim_get_cavities: NULL argument");
    *n = s->ncav;
    const int m = s->ncav < cap ? s->ncav : cap;
    if (m > 0 && host_out) {
        static_assert(sizeof(sim_cavity_t) == sizeof(Cav), "cavity layout");
        cudaMemcpyAsync(host_out, s->d_cav, sizeof(Cav) * (size_t)m, cudaMemcpyDeviceToHost, s->stream);
        if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_get_cavities");
    }
    return SIM_OK;
}

int sim_cavity_stats(const sim_t* s, double* phi_target, double* phi_achieved)
{
    if (!s) return SIM_ERR_ARG;
    if (phi_target) *phi_target = s->phi_target;
    if (phi_achieved) *phi_achieved = s->phi_achieved;
    return SIM_OK;
}

int sim_redo_count(sim_t* s, long long* n)
{
    if (!s || !n) return fail(s, SIM_ERR_ARG, "sim_redo_count: NULL argument");
    Ctl c;
    cudaMemcpyAsync(&c, s->ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_redo_count");
    *n = c.redo;
    return SIM_OK;
}

int sim_set_variant(sim_t* s, int variant, int use_graph)
{
    if (!s || (variant != SIM_VARIANT_UNFUSED && variant != SIM_VARIANT_FUSED)) return fail(s, SIM_ERR_ARG, "sim_set_variant: bad argument");
    if (variant == SIM_VARIANT_FUSED && !s->tm_ok)
        return fail(s, SIM_ERR_CUDA, "sim_set_variant: the fused variant needs tensor maps (cuTensorMapEncodeTiled failed in sim_create); this handle runs SIM_VARIANT_UNFUSED only");
    s->variant = variant; s->use_graph = use_graph ? 1 : 0; s->cfl_valid = false;
    return SIM_OK;
}

int sim_sweep_geometry(const sim_t* s, int dir, int* seg, int* ramp, long long* nblocks)
{
    if (!s || (dir != 0 && dir != 1) || !seg || !ramp || !nblocks) return SIM_ERR_ARG;
    sweep_geometry(s->P, dir, seg, ramp, nblocks);
    return SIM_OK;
}

int sim_set_launch_mode(sim_t* s, int use_graph, int use_pdl)
{
    if (!s) return SIM_ERR_ARG;
    const int g = use_graph ? 1 : 0, p = use_pdl ? 1 : 0;
    if (p != s->use_pdl && s->gexec) { cudaStreamSynchronize(s->stream); cudaGraphExecDestroy(s->gexec); s->gexec = nullptr; s->graph_failed = false; }
    s->use_graph = g; s->use_pdl = p;
    return SIM_OK;
}

long long sim_launch_count(const sim_t* s) { return s ? s->launches : 0; }

int sim_device_layout(const sim_t* s, void** plane0, long long* plane_stride, int* pitch, int* x_offset, int* y_offset)
{
    if (!s) return SIM_ERR_ARG;
    if (plane0) *plane0 = s->A;
    if (plane_stride) *plane_stride = s->P.fstride;
    if (pitch) *pitch = s->P.pitch;
    if (x_offset) *x_offset = NGX;
    if (y_offset) *y_offset = NGY;
    return SIM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// slab decomposition along x (include/nmsdt.h sim_slab_*)
// ---------------------------------------------------------------------------------------------------------------
namespace {
// input plane set of a pass of the current step: pass 1 reads A, pass 2 reads B
double* slab_pass_input(sim* s, int pass) { return pass == 1 ? s->A : s->B; }
int slab_dir(const sim* s, int pass) { const int d1 = (s->host_step & 1) ? 1 : 0; return pass == 1 ? d1 : 1 - d1; }
// the two edge columns (ghost = false) or ghost columns (ghost = true) of one x side of a plane set, rows 0..ny-1
SlabView slab_cols(double* plane0, long long fstride, int pitch, int nx, int side, bool ghost)
{
    const int col = side == 0 ? (ghost ? -NG : 0) : (ghost ? nx : nx - NG);
    return SlabView{plane0 + (long long)NGY * pitch + NGX + col, fstride, (long long)pitch};
}
int slab_args(sim* s, int pass, int side, const char* what)
{
    if (!s || (pass != 1 && pass != 2) || (side != 0 && side != 1)) return fail(s, SIM_ERR_ARG, std::string(what) + ": bad argument");
    if (!s->inited) return fail(s, SIM_ERR_STATE, std::string(what) + ": not initialised");
    if (s->variant != SIM_VARIANT_FUSED) return fail(s, SIM_ERR_STATE, std::string(what) + ": the slab calls drive the fused variant only");
    if (s->g.nx < NG) return fail(s, SIM_ERR_ARG, std::string(what) + ": a slab needs at least 2 columns");
    return SIM_OK;
}
} // namespace

size_t sim_slab_halo_bytes(const sim_t* s) { return s ? (size_t)7 * s->g.ny * NG * sizeof(double) : 0; }

int sim_slab_begin(sim_t* s, double dt_fixed)
{
    if (int rc = slab_args(s, 1, 0, "sim_slab_begin")) return rc;
    if (dt_fixed < 0.0) return fail(s, SIM_ERR_ARG, "sim_slab_begin: dt_fixed must be >= 0");
    launch_set_double(&s->ctl->dt_fixed, dt_fixed, s->stream);
    { KTimer t(s, SIM_K_CFL); launch_cfl(s->P, s->A, s->ctl, s->stream); }
    s->launches += 2;
    s->cfl_valid = false;           // sim_step after a slab-driven step recomputes its own dt
    return check_cuda(s, "sim_slab_begin");
}

int sim_slab_smax_ptr(sim_t* s, void** device_word)
{
    if (!s || !device_word) return fail(s, SIM_ERR_ARG, "sim_slab_smax_ptr: NULL argument");
    *device_word = &s->ctl->smax_bits;
    return SIM_OK;
}

int sim_slab_ctl(sim_t* s, int advance)
{
    if (int rc = slab_args(s, 1, 0, "sim_slab_ctl")) return rc;
    { KTimer t(s, SIM_K_CFL); launch_ctl(s->P, s->ctl, advance ? 1 : 0, s->stream); }
    s->launches++;
    if (advance) s->host_step++;
    return check_cuda(s, "sim_slab_ctl");
}

int sim_slab_pass_dir(const sim_t* s, int pass)
{
    if (!s || (pass != 1 && pass != 2)) return SIM_ERR_ARG;
    return slab_dir(s, pass);
}

int sim_slab_pass(sim_t* s, int pass)
{
    if (int rc = slab_args(s, pass, 0, "sim_slab_pass")) return rc;
    const int d = slab_dir(s, pass);
    double *in = slab_pass_input(s, pass), *out = pass == 1 ? s->B : s->A;
    { KTimer t(s, SIM_K_HALO); launch_halo(s->P, in, s->inflow, d, s->stream); }
    { KTimer t(s, d == 0 ? SIM_K_SWEEP_X : SIM_K_SWEEP_Y); launch_sweep_fused(s->P, in, pass == 1 ? &s->tmA : &s->tmB, out, &s->ctl->dt, s->ctl, d, pass, s->stream); }
    s->launches += 2;
    return check_cuda(s, "sim_slab_pass");
}

int sim_slab_pack(sim_t* s, int pass, int side, void* device_out)
{
    if (int rc = slab_args(s, pass, side, "sim_slab_pack")) return rc;
    if (!device_out) return fail(s, SIM_ERR_ARG, "sim_slab_pack: NULL buffer");
    const SlabView src = slab_cols(slab_pass_input(s, pass), s->P.fstride, s->P.pitch, s->g.nx, side, false);
    const SlabView dst{(double*)device_out, (long long)NG * s->g.ny, (long long)NG};
    { KTimer t(s, SIM_K_HALO); launch_slab_move(src, dst, s->g.ny, s->stream); }
    s->launches++;
    return check_cuda(s, "sim_slab_pack");
}

int sim_slab_unpack(sim_t* s, int pass, int side, const void* device_in)
{
    if (int rc = slab_args(s, pass, side, "sim_slab_unpack")) return rc;
    if (!device_in) return fail(s, SIM_ERR_ARG, "sim_slab_unpack: NULL buffer");
    const SlabView src{(double*)device_in, (long long)NG * s->g.ny, (long long)NG};
    const SlabView dst = slab_cols(slab_pass_input(s, pass), s->P.fstride, s->P.pitch, s->g.nx, side, true);
    { KTimer t(s, SIM_K_HALO); launch_slab_move(src, dst, s->g.ny, s->stream); }
    s->launches++;
    return check_cuda(s, "sim_slab_unpack");
}

int sim_slab_info(const sim_t* s, sim_slab_peer_t* out)
{
    if (!s || !out) return SIM_ERR_ARG;
    out->plane0[0] = s->A; out->plane0[1] = s->B;
    out->plane_stride = s->P.fstride; out->pitch = s->P.pitch; out->nx = s->g.nx; out->ny = s->g.ny;
    return SIM_OK;
}

int sim_slab_connect(sim_t* s, int side, const sim_slab_peer_t* peer)
{
    if (!s || (side != 0 && side != 1)) return fail(s, SIM_ERR_ARG, "sim_slab_connect: bad argument");
    if (!peer) { s->peer_on[side] = false; return SIM_OK; }
    if (!peer->plane0[0] || !peer->plane0[1] || peer->ny != s->g.ny || peer->nx < NG || peer->pitch < NGX + peer->nx + NG ||
        peer->plane_stride < (long long)peer->pitch * (peer->ny + 2 * NGY))
        return fail(s, SIM_ERR_ARG, "sim_slab_connect: neighbour layout does not fit (same ny, >= 2 columns)");
    s->peer[side] = *peer; s->peer_on[side] = true;
    return SIM_OK;
}

int sim_slab_push(sim_t* s, int pass)
{
    if (int rc = slab_args(s, pass, 0, "sim_slab_push")) return rc;
    const int k = pass == 1 ? 0 : 1;
    for (int side = 0; side < 2; ++side) {
        if (!s->peer_on[side]) continue;
        const sim_slab_peer_t& p = s->peer[side];
        // my x-lo edge columns are the x-hi ghost columns of my x-lo neighbour, and the other way round
        const SlabView src = slab_cols(slab_pass_input(s, pass), s->P.fstride, s->P.pitch, s->g.nx, side, false);
        const SlabView dst = slab_cols((double*)p.plane0[k], p.plane_stride, p.pitch, p.nx, 1 - side, true);
        { KTimer t(s, SIM_K_HALO); launch_slab_move(src, dst, s->g.ny, s->stream); }
        s->launches++;
    }
    return check_cuda(s, "sim_slab_push");
}

int sim_slab_ipc_export(const sim_t* s, void* host_handle64, size_t* offset_A, size_t* offset_B)
{
    if (!s || !host_handle64 || !offset_A || !offset_B) return SIM_ERR_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "ipc handle size");
    if (!s->owns) return fail(const_cast<sim*>(s), SIM_ERR_STATE, "sim_slab_ipc_export: needs a library-allocated workspace (device_buf = NULL)");
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, s->base) != cudaSuccess) return check_cuda(const_cast<sim*>(s), "sim_slab_ipc_export");
    std::memcpy(host_handle64, &h, 64);
    *offset_A = s->L.off_A; *offset_B = s->L.off_B;
    return SIM_OK;
}

int sim_slab_ipc_open(const void* host_handle64, void** device_base)
{
    if (!host_handle64 || !device_base) return SIM_ERR_ARG;
    cudaIpcMemHandle_t h; std::memcpy(&h, host_handle64, 64);
    if (cudaIpcOpenMemHandle(device_base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) return check_cuda(nullptr, "sim_slab_ipc_open");
    return SIM_OK;
}

int sim_slab_ipc_close(void* device_base)
{
    if (!device_base) return SIM_ERR_ARG;
    if (cudaIpcCloseMemHandle(device_base) != cudaSuccess) return check_cuda(nullptr, "sim_slab_ipc_close");
    return SIM_OK;
}

int sim_profile(sim_t* s, int on)
{
    if (!s) return SIM_ERR_ARG;
    if (on) {
        for (int k = 0; k < SIM_K_NKIND; ++k) { s->kms[k] = 0.0; s->kcount[k] = 0; }
        s->ev_used = 0;
        s->profile = true;
        return SIM_OK;
    }
    s->profile = false;
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_profile");
    for (size_t i = 0; i < s->ev_used; ++i) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, s->ev[i].a, s->ev[i].b) == cudaSuccess) { s->kms[s->ev[i].kind] += ms; s->kcount[s->ev[i].kind]++; }
    }
    s->ev_used = 0;
    return check_cuda(s, "sim_profile");
}

int sim_kernel_time(const sim_t* s, int kind, double* ms_total, long long* launches)
{
    if (!s || kind < 0 || kind >= SIM_K_NKIND || !ms_total || !launches) return SIM_ERR_ARG;
    *ms_total = s->kms[kind]; *launches = s->kcount[kind];
    return SIM_OK;
}

int sim_probe_fp64(sim_t* s, double* gflops_out, double* ms_out)
{
    if (!s || !gflops_out || !ms_out) return fail(s, SIM_ERR_ARG, "sim_probe_fp64: NULL argument");
    int rc = launch_probe_fp64(s->stream, gflops_out, ms_out);
    if (rc) return fail(s, SIM_ERR_CUDA, "sim_probe_fp64 failed");
    return SIM_OK;
}

int sim_probe_issue(sim_t* s, double ms_out[4])
{
    if (!s || !ms_out) return fail(s, SIM_ERR_ARG, "sim_probe_issue: NULL argument");
    if (launch_probe_issue(s->stream, ms_out)) return fail(s, SIM_ERR_CUDA, "sim_probe_issue failed");
    return SIM_OK;
}

namespace {
// library-owned scratch for the post-processing calls
double* post_scratch(sim* s, size_t bytes)
{
    if (bytes > s->post_bytes) {
        if (s->post) { cudaStreamSynchronize(s->stream); cudaFree(s->post); s->post = nullptr; s->post_bytes = 0; }
        if (cudaMalloc(&s->post, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        s->post_bytes = bytes;
    }
    return s->post;
}
} // namespace

int sim_profiles(sim_t* s, double p_front, double* host_pbar, double* host_rhobar, double* host_ubar, double* xs_out)
{
    if (!s) return fail(s, SIM_ERR_ARG, "sim_profiles: NULL handle");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_profiles: not initialised");
    double* buf = post_scratch(s, post_profiles_bytes(s->g.nx, s->g.ny));
    if (!buf) return fail(s, SIM_ERR_CUDA, "sim_profiles: cannot allocate scratch");
    double *d_out = nullptr, *d_xs = nullptr;
    s->launches += launch_profiles(s->P, s->A, p_front, buf, &d_out, &d_xs, s->stream);
    const size_t nb = (size_t)s->g.nx * sizeof(double);
    if (host_pbar) cudaMemcpyAsync(host_pbar, d_out, nb, cudaMemcpyDeviceToHost, s->stream);
    if (host_rhobar) cudaMemcpyAsync(host_rhobar, d_out + s->g.nx, nb, cudaMemcpyDeviceToHost, s->stream);
    if (host_ubar) cudaMemcpyAsync(host_ubar, d_out + 2 * (size_t)s->g.nx, nb, cudaMemcpyDeviceToHost, s->stream);
    if (xs_out) cudaMemcpyAsync(xs_out, d_xs, sizeof(double), cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_profiles");
    return check_cuda(s, "sim_profiles");
}

int sim_qdot_pdf(sim_t* s, double n_lo, double dn, int nbins, double* host_mass, long long* host_count)
{
    if (!s || !(dn > 0.0) || nbins < 1 || nbins > POST_MAX_BINS) return fail(s, SIM_ERR_ARG, "sim_qdot_pdf: bad argument (1 <= nbins <= 1024, dn > 0)");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_qdot_pdf: not initialised");
    if (!s->P.reactive) {                       // inert run: no energy release, empty statistics
        for (int b = 0; b < nbins; ++b) { if (host_mass) host_mass[b] = 0.0; if (host_count) host_count[b] = 0; }
        return SIM_OK;
    }
    double* buf = post_scratch(s, post_hist_bytes(nbins));
    if (!buf) return fail(s, SIM_ERR_CUDA, "sim_qdot_pdf: cannot allocate scratch");
    double* d_mass = nullptr; unsigned long long* d_count = nullptr;
    s->launches += launch_qdot_hist(s->P, s->A, n_lo, dn, nbins, buf, &d_mass, &d_count, s->stream);
    if (host_mass) cudaMemcpyAsync(host_mass, d_mass, sizeof(double) * nbins, cudaMemcpyDeviceToHost, s->stream);
    if (host_count) cudaMemcpyAsync(host_count, d_count, sizeof(long long) * nbins, cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_qdot_pdf");
    return check_cuda(s, "sim_qdot_pdf");
}

int sim_qdot_pdf_noalloc(sim_t* s, double n_lo, double dn, int nbins, double* host_mass, long long* host_count)
{
    if (!s || !(dn > 0.0) || nbins < 1) return fail(s, SIM_ERR_ARG, "sim_qdot_pdf_noalloc: bad argument (nbins >= 1, dn > 0)");
    if (nbins > POST_NOALLOC_MAX_BINS)
        return fail(s, SIM_ERR_ARG, "sim_qdot_pdf_noalloc: nbins = " + std::to_string(nbins) + " exceeds the " + std::to_string(POST_NOALLOC_MAX_BINS) +
                                    " bins of the library's static scratch; use sim_qdot_pdf (which allocates) for wider windows");
    if (!s->inited) return fail(s, SIM_ERR_STATE, "sim_qdot_pdf_noalloc: not initialised");
    if (!s->P.reactive) {                       // inert run: no energy release, empty statistics (as sim_qdot_pdf)
        for (int b = 0; b < nbins; ++b) { if (host_mass) host_mass[b] = 0.0; if (host_count) host_count[b] = 0; }
        return SIM_OK;
    }
    double* d_mass = nullptr; unsigned long long* d_count = nullptr;
    const char* why = "";
    const int n = launch_qdot_hist_noalloc(s->P, s->A, n_lo, dn, nbins, &d_mass, &d_count, s->stream, &why);
    if (n < 0) return fail(s, n == -1 ? SIM_ERR_ARG : SIM_ERR_CUDA, std::string("sim_qdot_pdf_noalloc: ") + why);
    s->launches += n;
    if (host_mass) cudaMemcpyAsync(host_mass, d_mass, sizeof(double) * nbins, cudaMemcpyDeviceToHost, s->stream);
    if (host_count) cudaMemcpyAsync(host_count, d_count, sizeof(long long) * nbins, cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_qdot_pdf_noalloc");
    return check_cuda(s, "sim_qdot_pdf_noalloc");
}

int sim_shock_kinematics(sim_t* s, const double* host_t, const double* host_xs, int n, double dtau, double* host_us, double* host_as)
{
    if (!s || !host_t || !host_xs || !host_us || !host_as || n < 2 || !(dtau > 0.0)) return fail(s, SIM_ERR_ARG, "sim_shock_kinematics: bad argument");
    double* buf = post_scratch(s, 4 * (size_t)n * sizeof(double));
    if (!buf) return fail(s, SIM_ERR_CUDA, "sim_shock_kinematics: cannot allocate scratch");
    const size_t nb = (size_t)n * sizeof(double);
    cudaMemcpyAsync(buf, host_t, nb, cudaMemcpyHostToDevice, s->stream);
    cudaMemcpyAsync(buf + n, host_xs, nb, cudaMemcpyHostToDevice, s->stream);
    s->launches += launch_kinematics(buf, buf + n, n, dtau, buf + 2 * (size_t)n, buf + 3 * (size_t)n, s->stream);
    cudaMemcpyAsync(host_us, buf + 2 * (size_t)n, nb, cudaMemcpyDeviceToHost, s->stream);
    cudaMemcpyAsync(host_as, buf + 3 * (size_t)n, nb, cudaMemcpyDeviceToHost, s->stream);
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return check_cuda(s, "sim_shock_kinematics");
    return check_cuda(s, "sim_shock_kinematics");
}

int sim_probe_math(sim_t* s, int fn, const double* host_x, int n, double a, double b, double* host_y0, double* host_y1)
{
    if (!s || !host_x || !host_y0 || !host_y1 || n < 1 || fn < 0 || fn > 8) return fail(s, SIM_ERR_ARG, "sim_probe_math: bad argument");
    if (launch_probe_math(s->P.pw, s->P.tab, fn, host_x, n, a, b, host_y0, host_y1, s->stream)) return fail(s, SIM_ERR_CUDA, "sim_probe_math failed");
    s->launches += 1;
    return SIM_OK;
}

} // extern "C"
