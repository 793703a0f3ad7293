// nmsdt_post.cu -- on-device post-processing of the state (readings R23-R26 of DESIGN.md), fp64, sm_100a:
//   k_prof_partial / k_prof_final / k_front : y-averaged profiles Eq. 9-11 and the leading-shock position of
//                                             Appendix C
//   k_qdot_hist / k_hist_final              : mass-weighted histogram of the volumetric energy-release rate, Eq. 14-16
//
//   k_kinematics                            : moving-averaged shock velocity / acceleration, Eq. C1-C2
// All sums have a fixed shape (no floating-point atomics): results are bit-identical from run to run.
// These passes read the state once (56 B/cell) and are not part of sim_step; with the fused path's own elementary
// functions (nmsdt_fast.cuh) the primitive recovery is cheap enough for them to be bound by HBM.
#include <mutex>
#include "nmsdt_host.h"
#include "nmsdt_fast.cuh"

namespace nmsdt {

namespace {

constexpr int PT = 128;            // threads per block of the profile kernels (one column per thread)

__device__ __forceinline__ void load_cell(const Params& P, const double* __restrict__ q, long long id, double c[7])
{
#pragma unroll
    for (int k = 0; k < 7; ++k) c[k] = q[k * P.fstride + id];
}

// partial column sums over the rows of one segment: part[(seg*3 + k)*nx + i], k = 0: p, 1: rho, 2: rho u
__global__ void __launch_bounds__(PT) k_prof_partial(const __grid_constant__ Params P, const double* __restrict__ q, double* __restrict__ part, int rows_per_seg)
{
    __shared__ __align__(16) double s_tab[MATH_TAB_DOUBLES];
    for (int k = threadIdx.x; k < MATH_TAB_DOUBLES; k += PT) s_tab[k] = P.tab[k];
    __syncthreads();
    const int i = blockIdx.x * PT + threadIdx.x;
    if (i >= P.nx) return;
    const int j0 = blockIdx.y * rows_per_seg, j1 = min(j0 + rows_per_seg, P.ny);
    double sp = 0.0, sr = 0.0, sm = 0.0;
    for (int j = j0; j < j1; ++j) {
        double c[7];
        load_cell(P, q, (long long)(j + NGY) * P.pitch + NGX + i, c);
        FCell W; double dE, q6n; bool hot = false;
        prim_cell<SRC_NONE>(P, s_tab, c, 0.0, 0.0, W, dE, q6n, hot);
        sp += W.p; sr += c[0] + c[1]; sm += c[2];
    }
    double* o = part + (size_t)blockIdx.y * 3 * P.nx + i;
    o[0] = sp; o[P.nx] = sr; o[2 * (size_t)P.nx] = sm;
}

// out[0..nx) = pbar, out[nx..2nx) = rhobar, out[2nx..3nx) = ubar; segments are added in order
__global__ void __launch_bounds__(PT) k_prof_final(const __grid_constant__ Params P, const double* __restrict__ part, int nseg, double* __restrict__ out)
{
    const int i = blockIdx.x * PT + threadIdx.x;
    if (i >= P.nx) return;
    double sp = 0.0, sr = 0.0, sm = 0.0;
    for (int s = 0; s < nseg; ++s) {
        const double* o = part + (size_t)s * 3 * P.nx + i;
        sp += o[0]; sr += o[P.nx]; sm += o[2 * (size_t)P.nx];
    }
    out[i] = sp / (double)P.ny;                       // Eq. 9
    out[P.nx + i] = sr / (double)P.ny;                // Eq. 10
    out[2 * (size_t)P.nx + i] = sm / sr;              // Eq. 11
}

// x_s = dx (1 + max{i : pbar_i >= p_front}), 0 if none (R25); one block
__global__ void __launch_bounds__(1024) k_front(const __grid_constant__ Params P, const double* __restrict__ pbar, double p_front, double* __restrict__ xs_out)
{
    __shared__ int s_best[32];
    int best = -1;
    for (int i = threadIdx.x; i < P.nx; i += blockDim.x)
        if (pbar[i] >= p_front) best = i;             // i increases along the loop
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if ((threadIdx.x & 31) == 0) s_best[threadIdx.x >> 5] = best;
    __syncthreads();
    if (threadIdx.x < 32) {
        best = threadIdx.x < (blockDim.x >> 5) ? s_best[threadIdx.x] : -1;
        for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
        if (threadIdx.x == 0) xs_out[0] = P.dx * (double)(best + 1);
    }
}

constexpr int HT = 256, HW = HT / 32;      // threads / warps per block of the histogram kernel

// Eq. 14-16.  Every warp owns whole rows (row = global warp id + k * number of warps) and a private histogram in shared
// memory; within a 32-cell group the lanes that fall into the same bin are added in lane order by shuffles and the sum
// is added by one lane, so the order of every floating-point addition is fixed by the launch shape alone.
__global__ void __launch_bounds__(HT, 4) k_qdot_hist(const __grid_constant__ Params P, const double* __restrict__ q, double n_lo, double dn, int nbins,
                                                  double* __restrict__ part_mass, unsigned long long* __restrict__ count)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    __shared__ __align__(16) double s_tab[MATH_TAB_DOUBLES_LOG];        // with the ln c_j part: Eq. 15 takes a logarithm
    for (int k = threadIdx.x; k < MATH_TAB_DOUBLES_LOG; k += HT) s_tab[k] = P.tab[k];
    double* s_mass = reinterpret_cast<double*>(s_raw);                         // [HW][nbins]
    int* s_cnt = reinterpret_cast<int*>(s_raw + (size_t)HW * nbins * sizeof(double));   // [HW][nbins]
    for (int k = threadIdx.x; k < HW * nbins; k += HT) { s_mass[k] = 0.0; s_cnt[k] = 0; }
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* wm = s_mass + (size_t)warp * nbins;
    int* wc = s_cnt + (size_t)warp * nbins;
    const double dA = P.dx * P.dy;
    const int gw = blockIdx.x * HW + warp, nw = gridDim.x * HW;
    for (int j = gw; j < P.ny; j += nw) {
        const long long row = (long long)(j + NGY) * P.pitch + NGX;
        for (int i0 = 0; i0 < P.nx; i0 += 32) {
            const int i = i0 + lane;
            int bin = -1;
            double mass = 0.0;
            if (i < P.nx) {
                double c[7];
                load_cell(P, q, row + i, c);
                FCell W; double dE, q6n; bool hot = false;
                prim_cell<SRC_NONE>(P, s_tab, c, 0.0, 0.0, W, dE, q6n, hot);
                const double T2 = cell_T2(P, W);
                if (T2 > 0.0) {
                    const double qdot = c[6] * P.Cpre * q_exp_neg(s_tab, P.Ta * q_rcp(T2)) * P.Q;      // Eq. 14 [W/m^3]
                    if (qdot > 1e-290) {                                                 // (a flushed exponential is far below any window)
                        const double n = q_log(s_tab, qdot * 1e-9) * 0.43429448190325182765;          // Eq. 15: log10 of GW/m^3
                        const double fb = floor((n - n_lo) / dn);
                        if (fb >= 0.0 && fb < (double)nbins) { bin = (int)fb; mass = c[1] * dA; }
                    }
                }
            }
            unsigned todo = __ballot_sync(0xffffffffu, bin >= 0);
            while (todo) {
                const int leader = __ffs(todo) - 1;
                const int b = __shfl_sync(0xffffffffu, bin, leader);
                unsigned peers = __ballot_sync(0xffffffffu, bin == b);
                todo &= ~peers;
                double s = 0.0;
                const int n = __popc(peers);
                while (peers) {                                   // lane order
                    const int src = __ffs(peers) - 1;
                    s += __shfl_sync(0xffffffffu, mass, src);
                    peers &= peers - 1;
                }
                if (lane == leader) { wm[b] += s; wc[b] += n; }
                __syncwarp();
            }
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += HT) {                // warps in order
        double s = 0.0; int n = 0;
        for (int w = 0; w < HW; ++w) { s += s_mass[(size_t)w * nbins + b]; n += s_cnt[(size_t)w * nbins + b]; }
        part_mass[(size_t)blockIdx.x * nbins + b] = s;
        if (n) atomicAdd(&count[b], (unsigned long long)n);        // integer: order independent
    }
}

__global__ void __launch_bounds__(256) k_hist_final(const double* __restrict__ part_mass, int nblocks, int nbins, double* __restrict__ mass)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nbins) return;
    double s = 0.0;
    for (int k = 0; k < nblocks; ++k) s += part_mass[(size_t)k * nbins + b];   // blocks in order
    mass[b] = s;
}

// x_s(tq) by linear interpolation between the samples that bracket tq (first bracket from the left)
__device__ __forceinline__ double interp_linear(const double* __restrict__ t, const double* __restrict__ x, int n, double tq, bool& ok)
{
    if (!(tq >= t[0]) || !(tq <= t[n - 1])) { ok = false; return 0.0; }
    int lo = 0, hi = n - 2;                          // smallest k in [0, n-2] with t[k+1] >= tq
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (t[mid + 1] < tq) lo = mid + 1; else hi = mid;
    }
    const double w = (tq - t[lo]) / (t[lo + 1] - t[lo]);
    return x[lo] + w * (x[lo + 1] - x[lo]);
}

__global__ void __launch_bounds__(128) k_kinematics(const double* __restrict__ t, const double* __restrict__ xs, int n, double dtau, double* __restrict__ us,
                                                    double* __restrict__ as)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);
    bool ok = true;
    const double xp = interp_linear(t, xs, n, t[k] + 0.5 * dtau, ok), xm = interp_linear(t, xs, n, t[k] - 0.5 * dtau, ok);
    us[k] = ok ? __ddiv_rn(__dsub_rn(xp, xm), dtau) : nan;                                       // Eq. C1
    ok = true;
    const double xpp = interp_linear(t, xs, n, t[k] + dtau, ok), xmm = interp_linear(t, xs, n, t[k] - dtau, ok);
    as[k] = ok ? __ddiv_rn(__dadd_rn(__dsub_rn(xpp, __dmul_rn(2.0, xs[k])), xmm), __dmul_rn(dtau, dtau)) : nan;   // Eq. C1 in C2
}

} // namespace

// ---------------------------------------------------------------------------------------------------------------
// launchers.  `buf` is device scratch of at least post_scratch_bytes(...) bytes; results are left on the device at the
// returned offsets (in doubles) and copied out by the C entry points.
// ---------------------------------------------------------------------------------------------------------------
static int prof_nseg(int nx, int ny)
{
    const int colblocks = (nx + PT - 1) / PT;
    int nseg = (8 * 148 + colblocks - 1) / colblocks;          // ~8 blocks per SM in total
    const int max_seg = (ny + 7) / 8;                          // at least 8 rows per segment
    if (nseg > max_seg) nseg = max_seg;
    if (nseg < 1) nseg = 1;
    return nseg;
}

size_t post_profiles_bytes(int nx, int ny) { return ((size_t)prof_nseg(nx, ny) * 3 + 3) * nx * sizeof(double) + 256; }

size_t post_hist_bytes(int nbins) { return ((size_t)POST_HIST_BLOCKS * nbins + 2 * (size_t)nbins) * sizeof(double) + 256; }

// profiles: out (device) = buf + 0: [pbar | rhobar | ubar] (3 nx doubles), then x_s (1 double, 256-byte aligned slot after them)
int launch_profiles(const Params& P, const double* q, double p_front, double* buf, double** d_out, double** d_xs, cudaStream_t s)
{
    const int nseg = prof_nseg(P.nx, P.ny);
    const int rows_per_seg = (P.ny + nseg - 1) / nseg;
    const int nseg_used = (P.ny + rows_per_seg - 1) / rows_per_seg;
    double* out = buf;
    double* xs = buf + 3 * (size_t)P.nx;
    double* part = xs + 32;
    dim3 grid((P.nx + PT - 1) / PT, nseg_used);
    k_prof_partial<<<grid, PT, 0, s>>>(P, q, part, rows_per_seg);
    k_prof_final<<<(P.nx + PT - 1) / PT, PT, 0, s>>>(P, part, nseg_used, out);
    k_front<<<1, 1024, 0, s>>>(P, out, p_front, xs);
    *d_out = out; *d_xs = xs;
    return 3;
}

// histogram: mass (device, nbins doubles) and count (device, nbins unsigned long long)
int launch_qdot_hist(const Params& P, const double* q, double n_lo, double dn, int nbins, double* buf, double** d_mass,
                     unsigned long long** d_count, cudaStream_t s)
{
    double* mass = buf;
    unsigned long long* count = reinterpret_cast<unsigned long long*>(buf + nbins);
    double* part = buf + 2 * (size_t)nbins;
    const size_t smem = (size_t)HW * nbins * (sizeof(double) + sizeof(int));
    static bool attr_set = false;
    if (!attr_set) { cudaFuncSetAttribute(k_qdot_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(HW * POST_MAX_BINS * 12)); attr_set = true; }
    cudaMemsetAsync(count, 0, sizeof(unsigned long long) * nbins, s);
    k_qdot_hist<<<POST_HIST_BLOCKS, HT, smem, s>>>(P, q, n_lo, dn, nbins, part, count);
    k_hist_final<<<(nbins + 255) / 256, 256, 0, s>>>(part, POST_HIST_BLOCKS, nbins, mass);
    *d_mass = mass; *d_count = count;
    return 2;
}

int launch_kinematics(const double* d_t, const double* d_xs, int n, double dtau, double* d_us, double* d_as, cudaStream_t s)
{
    k_kinematics<<<(n + 127) / 128, 128, 0, s>>>(d_t, d_xs, n, dtau, d_us, d_as);
    return 1;
}

} // namespace nmsdt

// ---------------------------------------------------------------------------------------------------------------
// sim_qdot_pdf_noalloc: the Eq. 14-16 histogram with its scratch in the library image instead of on the heap.
//
// Who needs it.  sim_qdot_pdf grows a per-handle scratch buffer with cudaMalloc / cudaFree on demand.  That is no use to
// a host program that has handed every byte of the GPU to its own arena (a solver that lends this library its workspace
// through sim_create's device_buf and has nothing left over for the driver's heap; cudaMalloc then fails although the
// arena has room), nor to an in-situ monitor that samples the histogram every few steps next to sim_step calls queued
// on other streams: cudaMalloc and cudaFree synchronise the whole device and would drain those queues at every sample.
// For them the scratch is the fixed array below: it is part of libnmsdt.so's device image, so EVERY GPU on which the
// library's kernels are loaded carries these ~2.3 MiB from that moment until the process exits, whether or not this entry
// point is ever called.  That is why the limit is modest: POST_NOALLOC_MAX_BINS = 512 bins (the paper's window, P:317,
// has 400); wider windows go through sim_qdot_pdf.
//
// Layout of the array (doubles): [0, nbins) mass, [nbins, 2 nbins) counts as unsigned 64-bit, then one row of nbins
// partial masses per block of k_qdot_hist -- the layout launch_qdot_hist gives its heap buffer.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_noalloc_hist_scratch[(size_t)nmsdt::POST_HIST_BLOCKS * nmsdt::POST_NOALLOC_MAX_BINS +
                                                                2 * (size_t)nmsdt::POST_NOALLOC_MAX_BINS];

namespace nmsdt {

namespace {
constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mutex;
double* g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};      // device address of the array on each ordinal, 0 = not looked up yet
}

// Returns the number of kernels enqueued, or -1 (argument) / -2 (CUDA) with *why pointing at a static message.
// In host code `g_noalloc_hist_scratch` is only the handle the runtime registered for the symbol: its device address
// differs per GPU and has to be asked for, once per device and with that device current (the first call on a device
// does it here, under a lock; it also raises the dynamic shared-memory limit of k_qdot_hist on that device).
int launch_qdot_hist_noalloc(const Params& P, const double* q, double n_lo, double dn, int nbins, double** d_mass, unsigned long long** d_count,
                             cudaStream_t s, const char** why)
{
    if (nbins < 1 || nbins > POST_NOALLOC_MAX_BINS) { *why = "nbins outside [1, 512]: the static scratch holds 512 bins, use sim_qdot_pdf for more"; return -1; }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { *why = cudaGetErrorString(e); cudaGetLastError(); return -2; }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) { *why = "device ordinal beyond the 64 this entry point keeps addresses for"; return -1; }
    cudaPointerAttributes at;
    e = cudaPointerGetAttributes(&at, q);
    if (e != cudaSuccess) { *why = cudaGetErrorString(e); cudaGetLastError(); return -2; }
    if (at.type != cudaMemoryTypeDevice || at.device != dev) { *why = "the device that holds the handle's state must be the current device"; return -1; }
    double* buf = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_addr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_noalloc_hist_scratch);
            if (e != cudaSuccess || !p) { *why = e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned NULL"; cudaGetLastError(); return -2; }
            e = cudaFuncSetAttribute(k_qdot_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(HW * POST_MAX_BINS * 12));
            if (e != cudaSuccess) { *why = cudaGetErrorString(e); cudaGetLastError(); return -2; }
            g_noalloc_addr[dev] = static_cast<double*>(p);
        }
        buf = g_noalloc_addr[dev];
    }
    double* mass = buf;
    unsigned long long* count = reinterpret_cast<unsigned long long*>(buf + nbins);
    double* part = buf + 2 * (size_t)nbins;
    const size_t smem = (size_t)HW * nbins * (sizeof(double) + sizeof(int));
    // The array keeps whatever the previous call (of any handle, any window) left in it.  Only the counts are accumulated
    // (integer atomics) and must start at zero; every block overwrites its whole row of partial masses and k_hist_final
    // overwrites the nbins masses, so nothing else of the old contents is ever read.
    cudaMemsetAsync(count, 0, sizeof(unsigned long long) * nbins, s);
    k_qdot_hist<<<POST_HIST_BLOCKS, HT, smem, s>>>(P, q, n_lo, dn, nbins, part, count);
    k_hist_final<<<(nbins + 255) / 256, 256, 0, s>>>(part, POST_HIST_BLOCKS, nbins, mass);
    *d_mass = mass; *d_count = count;
    return 2;
}

} // namespace nmsdt
