// nmsdt_step.cu -- time-step kernels of libnmsdt.so (fp64, sm_100a): halo fill (a2), Arrhenius source (a6),
// directional MUSCL-Hancock/HLLC sweeps (a4, a5), CFL reduction (a7).  See DESIGN.md for the kernel designs.
#include "nmsdt_host.h"

namespace nmsdt {

// ---------------------------------------------------------------------------------------------------------
// halo (a2; P:129 transmissive inflow, P:135 periodic top/bottom; R12)
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__global__ void k_halo(const __grid_constant__ Params P, double* __restrict__ q, const double* __restrict__ inflow)
{
    pdl_launch_dependents();
    pdl_wait();
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int f = blockIdx.y;                       // field
    double* a = q + (long long)f * P.fstride;
    if (DIR == 0) {
        if (t >= P.ny) return;
        double* row = a + (long long)(t + NGY) * P.pitch + NGX;
        const int nx = P.nx;
#pragma unroll
        for (int m = 1; m <= NG; ++m) {
            double v;
            switch (P.bc_xlo) {
                case 1:  v = row[((nx - m) % nx + nx) % nx]; break;
                case 2:  v = row[m - 1]; if (f == 2) v = -v; break;
                case 3:  v = inflow[f * P.ny + t]; break;
                default: v = row[0]; break;
            }
            double w;
            switch (P.bc_xhi) {
                case 1:  w = row[(m - 1) % nx]; break;
                case 2:  w = row[nx - m]; if (f == 2) w = -w; break;
                default: w = row[nx - 1]; break;
            }
            if (P.bc_xlo != 4) row[-m] = v;           // SIM_BC_EXTERNAL: the ghost columns belong to the neighbour slab
            if (P.bc_xhi != 4) row[nx - 1 + m] = w;
        }
    } else {
        if (t >= P.nx) return;
        double* col = a + (long long)NGY * P.pitch + NGX + t;
        const int ny = P.ny;
        const long long pt = P.pitch;
#pragma unroll
        for (int m = 1; m <= NG; ++m) {
            double v;
            switch (P.bc_ylo) {
                case 1:  v = col[(long long)(((ny - m) % ny + ny) % ny) * pt]; break;
                case 2:  v = col[(long long)(m - 1) * pt]; if (f == 3) v = -v; break;
                default: v = col[0]; break;
            }
            double w;
            switch (P.bc_yhi) {
                case 1:  w = col[(long long)((m - 1) % ny) * pt]; break;
                case 2:  w = col[(long long)(ny - m) * pt]; if (f == 3) w = -w; break;
                default: w = col[(long long)(ny - 1) * pt]; break;
            }
            col[-(long long)m * pt] = v;
            col[(long long)(ny - 1 + m) * pt] = w;
        }
    }
}

void launch_halo(const Params& P, double* q, const double* inflow, int dir, cudaStream_t s, bool pdl)
{
    const int n = dir == 0 ? P.ny : P.nx;
    dim3 grid((n + 127) / 128, 7);
    if (dir == 0) launch_k(k_halo<0>, grid, dim3(128), 0, s, pdl, P, q, inflow);
    else          launch_k(k_halo<1>, grid, dim3(128), 0, s, pdl, P, q, inflow);
}

// ---------------------------------------------------------------------------------------------------------
// standalone Arrhenius source step (a6), in place
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_source(const __grid_constant__ Params P, double* __restrict__ q,
                                                const double* __restrict__ dtp, double scale)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    if (i >= P.nx) return;
    const double tau = scale * (*dtp);
    const long long id = (long long)(j + NGY) * P.pitch + NGX + i;
    double c[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) c[k] = q[k * P.fstride + id];
    source_cell(P, c, tau);
    q[4 * P.fstride + id] = c[4];
    q[6 * P.fstride + id] = c[6];
}

void launch_source(const Params& P, double* q, const double* dtp, double scale, cudaStream_t s)
{
    dim3 grid((P.nx + 127) / 128, P.ny);
    k_source<<<grid, 128, 0, s>>>(P, q, dtp, scale);
}

// ---------------------------------------------------------------------------------------------------------
// directional sweep, register-marching form: one thread owns one line (DIR = 1: a column, coalesced across the
// warp; DIR = 0: a row) and marches along the sweep axis keeping the 3-cell primitive window, the previous
// face state and the previous flux in registers.  Nothing is recomputed except 4 ramp-up cells per segment.
// ---------------------------------------------------------------------------------------------------------
template <int DIR>
__global__ void __launch_bounds__(128) k_sweep_march(const __grid_constant__ Params P, const double* __restrict__ qin,
                                                     double* __restrict__ qout, const double* __restrict__ dtp, int seg)
{
    const int line = blockIdx.x * blockDim.x + threadIdx.x;
    const int nlines = DIR == 0 ? P.ny : P.nx;
    const int n = DIR == 0 ? P.nx : P.ny;
    if (line >= nlines) return;
    const int c0 = blockIdx.y * seg;
    const int c1 = min(c0 + seg, n);
    const double dtdx = (*dtp) / (DIR == 0 ? P.dx : P.dy);
    const long long stride = DIR == 0 ? 1 : P.pitch;
    const long long base = DIR == 0 ? (long long)(line + NGY) * P.pitch + NGX : (long long)NGY * P.pitch + NGX + line;
    constexpr int kn = DIR == 0 ? 2 : 3, kt = DIR == 0 ? 3 : 2;
    const long long fs = P.fstride;

    Prim Wm, W0, Wp;
    double rho0 = 1.0, c20 = 1.0, rhop, c2p;
    Face prevR;
    double prevF[7], prevU = 0.0;
    Wm = W0 = Prim{1, 1, 0, 0, 1, 0.5, 0};
    prevR = Face{1, 1, 0, 0, 1, 0.5, 0, 1, 1, 1};
#pragma unroll
    for (int k = 0; k < 7; ++k) prevF[k] = 0.0;

    for (int c = c0 - 2; c < c1 + 2; ++c) {
        const long long id = base + (long long)c * stride;
        double q[7];
        q[0] = qin[id]; q[1] = qin[fs + id]; q[2] = qin[kn * fs + id]; q[3] = qin[kt * fs + id];
        q[4] = qin[4 * fs + id]; q[5] = qin[5 * fs + id]; q[6] = qin[6 * fs + id];
        cons_to_prim(P, q, Wp, rhop, c2p, nullptr);
        const int jj = c - (c0 - 2);
        if (jj >= 2) {   // centre cell c-1 has both neighbours
            double WL[7], WR[7];
            reconstruct(P, Wm, W0, Wp, rho0, c20, 0.5 * dtdx, WL, WR);
            if (jj >= 3) {
                Face fl;
                face_state(P, WL, fl);
                double F[7], uf;
                hllc(prevR, fl, F, uf);          // face between cells c-2 and c-1
                if (jj >= 4) {                   // update cell c-2
                    const long long iu = base + (long long)(c - 2) * stride;
                    double o[7];
                    o[0] = qin[iu]; o[1] = qin[fs + iu]; o[2] = qin[kn * fs + iu]; o[3] = qin[kt * fs + iu];
                    o[4] = qin[4 * fs + iu]; o[5] = qin[5 * fs + iu]; o[6] = qin[6 * fs + iu];
                    const double z1n = o[5];
#pragma unroll
                    for (int k = 0; k < 7; ++k) o[k] = o[k] - dtdx * (F[k] - prevF[k]);
                    o[5] = o[5] + dtdx * z1n * (uf - prevU);      // R8: non-conservative z1 term
                    o[5] = clampd(o[5], P.z_min, P.z_max);
                    qout[iu] = o[0]; qout[fs + iu] = o[1]; qout[kn * fs + iu] = o[2]; qout[kt * fs + iu] = o[3];
                    qout[4 * fs + iu] = o[4]; qout[5 * fs + iu] = o[5]; qout[6 * fs + iu] = o[6];
                }
#pragma unroll
                for (int k = 0; k < 7; ++k) prevF[k] = F[k];
                prevU = uf;
            }
            face_state(P, WR, prevR);
        }
        Wm = W0; W0 = Wp; rho0 = rhop; c20 = c2p;
    }
}

void launch_sweep_march(const Params& P, const double* qin, double* qout, const double* dtp, int dir, cudaStream_t s)
{
    const int nlines = dir == 0 ? P.ny : P.nx;
    const int n = dir == 0 ? P.nx : P.ny;
    const int seg = 64;
    dim3 grid((nlines + 127) / 128, (n + seg - 1) / seg);
    if (dir == 0) k_sweep_march<0><<<grid, 128, 0, s>>>(P, qin, qout, dtp, seg);
    else          k_sweep_march<1><<<grid, 128, 0, s>>>(P, qin, qout, dtp, seg);
}

// ---------------------------------------------------------------------------------------------------------
// CFL reduction (a7): S_max = max(max(|u|,|v|) + c); max is order independent -> bitwise deterministic
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_cfl(const __grid_constant__ Params P, const double* __restrict__ q, Ctl* ctl)
{
    double smax = 0.0;
    int bad = 0;
    const long long ncell = (long long)P.nx * P.ny;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < ncell; t += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(t / P.nx), i = (int)(t - (long long)j * P.nx);
        const long long id = (long long)(j + NGY) * P.pitch + NGX + i;
        double c[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) c[k] = q[k * P.fstride + id];
        Prim W; double rho, c2;
        cons_to_prim(P, c, W, rho, c2, nullptr);
        const double a = fmax(fabs(W.un), fabs(W.ut)) + sqrt(c2);
        smax = fmax(smax, a);
        const bool ok = isfinite(c[0]) && isfinite(c[1]) && isfinite(c[2]) && isfinite(c[3]) && isfinite(c[4]) && isfinite(c[5])
                        && isfinite(c[6]) && c[0] > 0.0 && c[1] > 0.0 && isfinite(a);
        bad |= ok ? 0 : 1;
    }
    for (int o = 16; o > 0; o >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    __shared__ double s_m[8];
    __shared__ int s_b[8];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { s_m[w] = smax; s_b[w] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { smax = fmax(smax, s_m[k]); bad |= s_b[k]; }
        atomicMax(&ctl->smax_bits, dbits(smax));
        if (bad) atomicOr(&ctl->bad, 1);
    }
}

void launch_cfl(const Params& P, const double* q, Ctl* ctl, cudaStream_t s)
{
    const long long ncell = (long long)P.nx * P.ny;
    int blocks = (int)((ncell + 255) / 256);
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_cfl<<<blocks, 256, 0, s>>>(P, q, ctl);
}

__global__ void k_finalize_dt(const __grid_constant__ Params P, Ctl* ctl)
{
    const double smax = __longlong_as_double((long long)ctl->smax_bits);
    ctl->dt = ctl->dt_fixed > 0.0 ? ctl->dt_fixed : P.cfl * P.hmin / smax;
    ctl->smax_bits = 0ull;
}
void launch_finalize_dt(const Params& P, Ctl* ctl, cudaStream_t s) { k_finalize_dt<<<1, 1, 0, s>>>(P, ctl); }

__global__ void k_advance(Ctl* ctl)
{
    ctl->t += ctl->dt;
    ctl->dt_last = ctl->dt;
    ctl->step += 1;
}
void launch_advance(Ctl* ctl, cudaStream_t s) { k_advance<<<1, 1, 0, s>>>(ctl); }

__global__ void k_set_double(double* p, double v) { *p = v; }
void launch_set_double(double* p, double v, cudaStream_t s) { k_set_double<<<1, 1, 0, s>>>(p, v); }

} // namespace nmsdt
