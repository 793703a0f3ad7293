/*
 * nmsdt_probe.h -- measurement probes exported by libnmsdt.so beside the C ABI of the method (include/nmsdt.h).
 *
 * None of these takes part in a time step.  bench.py uses sim_probe_fp64 / sim_probe_issue for the denominators of its
 * `roofline` block, tests/test_gpu_math.py uses sim_probe_math to check the fused path's own fp64
 * elementary functions against long-double references.  Their kernels live in csrc/nmsdt_probe.cu.  Conventions (return
 * codes, HOST pointers, [sync]) are those of nmsdt.h; the handle only supplies the stream and, for sim_probe_math, the
 * function tables of its equation of state.
 */
#ifndef NMSDT_PROBE_H
#define NMSDT_PROBE_H

#include "nmsdt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measured FP64 FMA throughput of this device in GFLOP/s (2 flop per DFMA), probe kernel of ~ms. [sync] */
int sim_probe_fp64(sim_t*, double* gflops_out, double* ms_out);
/* Issue-slot probe behind the roofline model of DESIGN.md section 6: times [ms] of a kernel of 8 independent DFMA chains
   per thread with 0, 4, 8 and 16 independent 32-bit ALU instructions interleaved per 8 DFMA, at the sweeps' residency
   (4 warps per scheduler).  ms_out[k]/ms_out[0] = 1, 1, 1, 1.5 would mean the other instructions hide under the
   half-rate FP64 pipe; 1, 1.25, 1.5, 2 means a DFMA holds the issue port for both of its cycles, so that a step
   costs 2 F + O issue slots (F FP64-pipe instructions, O others). [sync] */
int sim_probe_issue(sim_t*, double ms_out[4]);
/* Accuracy probe of the fused path's own fp64 elementary functions (the Cochran-Chan powers of Eq. 3-4, and
   the Arrhenius exponential of Eq. 6, are evaluated with these instead of the CUDA math library; DESIGN.md
   section 5).  Evaluates function `fn` on host_x[n] on the device and returns host_y0[n], host_y1[n] (HOST arrays,
   caller-owned; y1 is written with zeros when the function has one result):
     0: 1/x            1: sqrt(x)        2: ln(x)        3: (x^a, x^b)        4: exp(-x)
     5: (max(x,1), min(max(x,0),1))      6: (max(x,0), min(x,690))
     7: (x^C, x^D) for the handle's own Eq. 3 exponents by the table route of the step kernels (a, b ignored)
     8: (max(sqrt(x/a), 1), max(sqrt(a/x), 1)): the floored sound speed of R10 from rho c^2 and rho without a reciprocal
   x must be a positive normal number for 0-3. SIM_ERR_ARG on NULL / n < 1 / unknown fn. [sync] */
int sim_probe_math(sim_t*, int fn, const double* host_x, int n, double a, double b, double* host_y0, double* host_y1);

#ifdef __cplusplus
}
#endif
#endif
