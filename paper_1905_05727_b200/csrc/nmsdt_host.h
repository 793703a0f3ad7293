// nmsdt_host.h -- host-side declarations shared by the .cu files of libnmsdt.so (not part of the public ABI).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "nmsdt_device.cuh"

namespace nmsdt {

struct Cav { double x, y, r; };

struct Hug { double rho_s, U_s, u_p, T2_s, rho1_s; };

struct DiagOut {   // device-side result of the diagnostics reduction
    double sum[7]; // q0..q4, q6, rate
    double smax;
    int bad;
    int pad;
};

constexpr int DIAG_BLOCKS = 1184;          // 8 x 148
constexpr int DIAG_NV = 8;                 // 7 sums + smax

// kernel launch with (pdl = true) or without the programmatic-stream-serialization attribute (see pdl_wait, nmsdt_device.cuh)
template <typename... KArgs, typename... Args>
inline cudaError_t launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// step kernels (nmsdt_step.cu)
void launch_halo(const Params& P, double* q, const double* inflow, int dir, cudaStream_t s, bool pdl = false);
void launch_source(const Params& P, double* q, const double* dtp, double scale, cudaStream_t s);
void launch_sweep_march(const Params& P, const double* qin, double* qout, const double* dtp, int dir, cudaStream_t s);
void launch_cfl(const Params& P, const double* q, Ctl* ctl, cudaStream_t s);
void launch_finalize_dt(const Params& P, Ctl* ctl, cudaStream_t s);
void launch_advance(Ctl* ctl, cudaStream_t s);
void launch_set_double(double* p, double v, cudaStream_t s);
int  launch_probe_fp64(cudaStream_t s, double* gflops, double* ms);
int  launch_probe_issue(cudaStream_t s, double ms[4]);

// fused production path (nmsdt_fused.cu). dtp -> {dt (or tau for the source kernel), tsafe}; mode 0 plain, 1 leading
// source on load, 2 trailing source + max-wavespeed partial
void init_fused_kernels();
// end_step (pass 2 only): the last block to finish also ends the step (t, step counter, next dt: what k_ctl does otherwise)
// tm_in: tensor map of the plane set qin (dims {pitch, rows, 7}, box {32, 1, 7}; make_plane_tensor_map in nmsdt_capi.cu)
void launch_sweep_fused(const Params& P, const double* qin, const CUtensorMap* tm_in, double* qout, const double* dtp, Ctl* ctl, int dir, int mode,
                        cudaStream_t s, bool pdl = false, bool end_step = false);
void launch_source_fast(const Params& P, double* q, const double* dtp, cudaStream_t s);
void sweep_geometry(const Params& P, int dir, int* seg, int* ramp, long long* nblocks);
void launch_ctl(const Params& P, Ctl* ctl, int advance, cudaStream_t s, bool pdl = false);
double host_tsafe(double tau, double Cpre, double Ta, double theta0);
int  launch_probe_math(const PowCoef& pw, const double* tab_dev, int fn, const double* host_x, int n, double a, double b, double* host_y0, double* host_y1,
                       cudaStream_t s);

// post-processing (nmsdt_post.cu): Eq. 9-11 profiles + front position, Eq. 14-16 histogram, Eq. C1-C2 kinematics.
// Each launcher returns the number of kernels it enqueued.
constexpr int POST_HIST_BLOCKS = 592;      // 4 x 148
constexpr int POST_MAX_BINS = 1024;
size_t post_profiles_bytes(int nx, int ny);
size_t post_hist_bytes(int nbins);
int launch_profiles(const Params& P, const double* q, double p_front, double* buf, double** d_out, double** d_xs, cudaStream_t s);
int launch_qdot_hist(const Params& P, const double* q, double n_lo, double dn, int nbins, double* buf, double** d_mass,
                     unsigned long long** d_count, cudaStream_t s);
int launch_kinematics(const double* d_t, const double* d_xs, int n, double dtau, double* d_us, double* d_as, cudaStream_t s);
// sim_qdot_pdf_noalloc: the same two kernels on a fixed __device__ array of nmsdt_post.cu (no heap); -1 / -2 + *why on error
constexpr int POST_NOALLOC_MAX_BINS = 512;
int launch_qdot_hist_noalloc(const Params& P, const double* q, double n_lo, double dn, int nbins, double** d_mass, unsigned long long** d_count,
                             cudaStream_t s, const char** why);

// slab decomposition (nmsdt_slab.cu): a block of 7 planes x ny rows x 2 columns inside some strided layout
struct SlabView { double* base; long long fstride; long long pitch; };
void launch_slab_move(const SlabView& src, const SlabView& dst, int ny, cudaStream_t s);

// init / output kernels (nmsdt_init.cu)
void launch_zero_plane(const Params& P, double* plane, cudaStream_t s);
void launch_clamp_z1(const Params& P, double* q5, cudaStream_t s);
void launch_shift_cavities(Cav* cav, int n, double shift, cudaStream_t s);
void launch_paint(const Params& P, double* prof_plane, const Cav* cav, int ncav, double h, cudaStream_t s);
void launch_fill_state(const Params& P, double* q, int shock_cells, Hug hug, double p_shock, double p0, double rho1_0,
                       double rho2_0, cudaStream_t s);
void launch_capture_inflow(const Params& P, const double* q, double* inflow, cudaStream_t s);
void launch_diag(const Params& P, const double* q, double* partial, DiagOut* out, cudaStream_t s);
void launch_derived(const Params& P, const double* q, int field_id, double* out_dense, cudaStream_t s);
// seeded generator on the device; returns number of cavities (<0 on error); list left in d_cav
int  generate_cavities(unsigned long long seed, double phi, double dmin, double dmax, double min_gap, int x_lo, int x_hi,
                       int ny, int periodic_y, Cav** d_cav_out, cudaStream_t s, long long* launches, long long* sum_r2_256,
                       long long* target_r2_256);

} // namespace nmsdt
