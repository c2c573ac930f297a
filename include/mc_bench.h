/* mc_bench.h -- C ABI of libmc_bench: the measurement instruments of bench.py.  NOT part of the product boundary
 * (include/mc.h, libmc.so): a user of the integrator never needs these.  Built by benchlib/build.py into
 * benchlib/libmc_bench.so; error codes are mc.h's mc_error (a failing CUDA call also prints its message to stderr). */
#ifndef MC_BENCH_H_
#define MC_BENCH_H_

#include "mc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* DFMA throughput of the device, measured: every SM runs independent FMA chains for about
 * `millis` ms; *out_tflops = 2 * FMAs / time (CUDA events).  The roofline denominator of bench.py
 * (MEASURED_PEAKS.json has no FP64 entry).  Synchronous. */
int mc_fp64_peak(int32_t device, double millis, double* out_tflops, double* out_sm_clock_mhz);

/* Operand bandwidth of the FP64 pipe, measured: a warp-wide FP64 instruction nominally
 * occupies a sub-partition's 16-lane pipe for 2 cycles, but the register file delivers one 64-bit operand per cycle,
 * so an FMA that reads three distinct vector registers takes 3.  kind selects the instruction the probe repeats
 * (8 independent accumulators per thread, 4 warps per sub-partition, about `millis` ms, best of 4):
 *   0: x <- fma(y, z, x), three distinct registers        2: x <- fma(y, c[bank], x), two registers + constant
 *   1: x <- fma(y, s, x), s reused by consecutive FMAs    3: x <- x * y (DMUL)
 * *out_cycles_per_warp_instr = SM cycles (at the device's maximum clock) per warp instruction per sub-partition;
 * *out_tflops (optional) = the corresponding flop rate of the whole device.  Synchronous.  MC_EINVAL: bad kind. */
int mc_fp64_probe(int32_t device, double millis, int32_t kind, double* out_cycles_per_warp_instr, double* out_tflops);

/* Algorithmic operation counts of the kernels' own formulation, per trajectory.
 * Host-only, needs no GPU: the library instantiates the math templates the kernels are built from
 * (csrc/mc_math.cuh, mc_correct.cuh) with a scalar type that counts its own operations, so the figures follow
 * the code.  fma = fused multiply-adds, mul, add (additions and subtractions), special = rsqrt + reciprocal +
 * division + sqrt (one each; the refinement steps around the hardware seeds are not algorithmic work).
 * flop = 2 fma + mul + add + special.  Operations on constants and negations are free.
 *   rhs            one evaluation of dz/dt (eqs 6-9)
 *   base_step      one uncorrected step of the base integrator, RHS evaluations included
 *   correct_fixed  the part of the correction done once per step: eq (10), L_t; for mode 2 the whole dual
 *                  scaling with newton_iters polynomial Newton iterations; 0 for mode 0
 *   gn_step        one Gauss-Newton step of mode 3 (gradient + H, 4 x 4 solve, update, termination test); else 0
 *   status         the |r|^2 test of a completed step
 *   references     E0, J0 of a state (H + J)
 *   renorm         one shadow renormalisation (distance, pull-back, eq 10, re-referenced integrals)
 * A trajectory-step costs base_step + correct_fixed + status + gn_step x (Gauss-Newton steps taken, mc_get_work).
 * With MC_TERM_RR the RHS, the base step and the renormalisation include the radiation-reaction force and the four
 * dissipation integrals (16 components per trajectory).
 * Errors: MC_EINVAL (null, unknown term bit / mode / integrator, newton_iters outside 1..16). */
typedef struct mc_op_counts { int64_t fma, mul, add, special; } mc_op_counts;
typedef struct mc_flop_model_t {
  mc_op_counts rhs, base_step, correct_fixed, gn_step, status, references, renorm;
} mc_flop_model_t;
int mc_flop_model(uint32_t terms, int32_t correction_mode, int32_t integrator, int32_t newton_iters,
                  mc_flop_model_t* out);

#ifdef __cplusplus
}
#endif
#endif /* MC_BENCH_H_ */
