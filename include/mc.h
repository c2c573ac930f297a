/* mc.h -- C ABI of libmc: batched manifold-corrected RK4 integration of the conservative PN
 * Hamiltonian of spinning compact binaries on one NVIDIA B200 (sm_100a), FP64 throughout.
 *
 * Method: arXiv 1802.00147 (cited below as PAPER.md:<line>, the text under /root/reference at build
 * time) as read in DESIGN.md (cited as DESIGN.md Rn).  No C++ types and no exceptions cross this
 * boundary; every function returns 0 (MC_OK) or a negative mc_error.  There is no CPU fallback.
 *
 * Data layout (all entry points): one orbit's state is z = (r, p, S1hat, S2hat), 12 doubles
 * (PAPER.md:81, 120): r in units of M, p in units of mu, unit spin vectors; G = c = M = 1.  A batch
 * is structure-of-arrays, double[12][n_orbits], row c holds component c of every orbit in the order
 * rx ry rz px py pz s1x s1y s1z s2x s2y s2z.
 */
#ifndef MC_H_
#define MC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mc_handle mc_handle; /* opaque; created by mc_create, freed by mc_destroy.  A handle owns device scratch
                                       (status, work queue, carry) that its calls reuse in stream order: use one
                                       handle per stream and do not call into one handle from two host threads at once */

enum mc_error {
  MC_OK = 0,
  MC_EINVAL = -1,  /* null pointer, negative size, unknown mode/term bit, beta outside (0,1], ... */
  MC_ECUDA = -2,   /* a CUDA runtime call failed; mc_strerror(MC_ECUDA) returns the CUDA message  */
  MC_EARCH = -3,   /* the device is not compute capability 10.x (the library holds sm_100a code only) */
  MC_ENOMEM = -4,  /* host allocation failed */
  MC_ELIMIT = -5   /* mc_integrate_static only: the batch exceeds MC_STATIC_MAX_TRAJECTORIES */
};

/* Hamiltonian terms, eq (1) of the paper.  H_N is always on. */
enum mc_terms {
  MC_TERM_1PN = 1u,   /* H_1PN (ADM; R1)                        */
  MC_TERM_2PN = 2u,   /* H_2PN                                            */
  MC_TERM_SO = 4u,    /* spin-orbit, L-terms of eqs (8)-(9) */
  MC_TERM_S1S2 = 8u,  /* eq (3)                              */
  MC_TERM_QM = 16u,   /* eqs (4)-(5), quadrupole-monopole */
  MC_TERM_RR = 32u    /* a_2.5PN of eq (6): leading-order radiation reaction in the ADM gauge
                         (R21; not printed in the paper).  NON-conservative: every trajectory also
                         carries the work W = int (dr/dt).a dt and the torque integral G = int r x a dt of the
                         force, and the correction (modes 2, 3) targets E0 + W and J0 + G, the "integral invariant
                         relation" of PAPER.md:221; see mc_get_dissipation.  Default off.  One combination is not
                         built: per_orbit = 1 together with MC_INTEG_RK5 (mc_integrate, and mc_eval with what = 3, return MC_EINVAL; the 45
                         per-orbit constants, six stages and 16 components exceed the 255-register budget and the
                         library ships no kernel that spills)                                               */
};

/* Correction applied after every RK4 step. */
enum mc_correction {
  MC_CORR_NONE = 0,      /* plain RK4                                                             */
  MC_CORR_SPINS = 1,     /* eq (10): S_i_hat <- S_i_hat / |S_i_hat|                                 */
  MC_CORR_DUAL = 2,      /* eq (10) + the paper's dual scaling p <- alpha p, r <- beta r, eqs (11)-(13):
                            exact H = E0 and |J| = |J0|                                            */
  MC_CORR_SIXINT = 3     /* eq (10) + minimal-norm projection of (r,p) onto H = E0, J = J0 (vector):
                            all six integrals to round-off (R4); "correction on"         */
};

/* Per-orbit outcome (merged / unbound orbits are dropped; R13). */
enum mc_status {
  MC_ST_OK = 0,
  MC_ST_MERGED = 1,     /* |r| < r_merge after a step; state frozen at the last good step */
  MC_ST_UNBOUND = 2,    /* |r| > r_escape                                                   */
  MC_ST_NONFINITE = 3,  /* a non-finite component in the orbit or its shadow                */
  MC_ST_NEWTON_FLAG = 256 /* OR-ed in: mode 2 skipped its (r,p) scaling on >= 1 step (R7) */
};

/* Base integrator (R9).  BASELINE.json fixes classical RK4; the paper itself says "RK5"
 * without a tableau, read as Butcher's six-stage fifth-order method. */
enum mc_integrator {
  MC_INTEG_RK4 = 0,   /* c = 0, 1/2, 1/2, 1; b = 1/6, 1/3, 1/3, 1/6                                        */
  MC_INTEG_RK5 = 1    /* c = 0, 1/4, 1/4, 1/2, 3/4, 1; b = 7/90, 0, 32/90, 12/90, 32/90, 7/90                */
};

typedef struct mc_params {
  uint32_t struct_size;   /* = sizeof(mc_params); checked by mc_create                                   */
  uint32_t terms;         /* OR of mc_terms                                                              */
  int32_t device;         /* CUDA device ordinal                                                         */
  int32_t per_orbit;      /* 0: the five scalars below apply to every orbit; 1: use the five device arrays;
                             2: beta, chi1, chi2 scalars for every orbit, kq1, kq2 per orbit from d_kq1, d_kq2
                             (BASELINE config 3: one binary model, a scan over quadrupole coefficients) -- the
                             constants that do not depend on kq stay constant-bank operands of the kernel      */
  double beta;            /* mass ratio m1/m2 in (0,1]                                       */
  double chi1, chi2;      /* dimensionless spins in [0,1]                                   */
  double kq1, kq2;        /* quadrupole coefficients, 1 = black hole (R16)         */
  const double* d_beta;   /* per_orbit = 1: DEVICE arrays of length >= n_orbits, owned by the caller,      */
  const double* d_chi1;   /*   must stay valid until mc_destroy; values are not validated on the device    */
  const double* d_chi2;
  const double* d_kq1;
  const double* d_kq2;
  int32_t renorm_interval; /* steps between shadow renormalisations, > 0 (BASELINE config 1: 100)          */
  int32_t newton_iters;    /* Newton iterations, 1..16 (R6): the cap of mode 3, the fixed count of
                              mode 2; default 4                                                             */
  double newton_tol;       /* epsilon of PAPER.md:197 (default 1e-10).  Mode 3: a Gauss-Newton step with
                              |(dr,dp)|_2 <= epsilon |p|_2 is the last one; 0 = always newton_iters steps.
                              Mode 2: the scaling is skipped unless the last |dv| <= epsilon               */
  double r_merge;          /* default 2    (R13)                                                 */
  double r_escape;         /* default 1e4                                                                  */
  void* cuda_stream;       /* cudaStream_t all work is enqueued on (e.g. torch's current stream); NULL = 0 */
  int32_t chunk_steps;     /* scheduling only, never changes a result bit: 0 = automatic; > 0 = the kernel's
                              work items are chunks of this many steps (state parked in device scratch owned
                              by the handle between chunks)                          */
  int32_t integrator;      /* mc_integrator; default MC_INTEG_RK4                                          */
  double wait_budget_s;    /* scheduling watchdog, default 600: the kernel is persistent and a warp may wait for the
                              previous chunk of its work unit, which another resident warp holds.  That cannot
                              deadlock as long as the WHOLE GRID IS CO-RESIDENT: the library sizes the grid with the
                              occupancy API on an otherwise idle device.  Under MPS / a co-tenant that takes SM
                              resources the assumption can fail; a wait longer than this many seconds then ends the
                              launch with a trap (MC_ECUDA on the next call) instead of a hang.  Raise it for
                              profiler replays or very long forced chunks (chunk_steps); must be in (0, 1e9]   */
  int32_t regroup;         /* scheduling only, never changes a result bit; 0 (default) or 1.  1: mc_integrate first
                              sorts the orbits by their energy H at t = 0 on the device (one small kernel + a
                              radix sort, stream-ordered) and lets slot s of the launch integrate the s-th orbit
                              in that order; inputs and outputs keep the caller's order.  Orbits of equal energy
                              have equal radial periods to 1PN order, so the 16 orbits of a warp keep passing
                              periastron together and need their second Gauss-Newton step at the same steps.
                              Pays for UNSTRUCTURED batches (random initial conditions: +7 %, DESIGN.md section
                              10); a grid scan in row-major order is already grouped and loses a few per cent.
                              Ignored with sampled output, by mc_integrate_ex and below 64 orbits             */
  int32_t reserved_;       /* 0                                                                            */
} mc_params;

/* Fill *p with defaults: terms = 1PN|2PN|SO|S1S2, device 0, uniform beta = chi = kq = 1,
 * renorm_interval 100, newton_iters 4, newton_tol 1e-10, r_merge 2, r_escape 1e4, stream NULL,
 * chunk_steps 0, integrator RK4, wait_budget_s 600, regroup 0. */
int mc_params_default(mc_params* p);

/* Validate params, select the device, allocate the handle.  *out_handle is set only on success. */
int mc_create(const mc_params* params, mc_handle** out_handle);

/* Integrate n_orbits independent orbits for n_steps steps of size step_h (may be negative) of the base
 * integrator (classical RK4 unless params.integrator says RK5), applying correction_mode after every
 * step (the per-orbit algorithm is spelled out in DESIGN.md section 2).  Reference integrals E0, J0 are taken from the input states
 * (PAPER.md:136); with correction_mode >= 1 the input spins are normalised first.
 *
 * shadow_eps != 0 adds, per orbit, a shadow trajectory started at rx + shadow_eps, integrated and
 * corrected onto its own integrals, renormalised to distance |shadow_eps| every renorm_interval
 * steps, and writes the fast Lyapunov indicator FLI = log10(d(t)/d(0)) (R10-R12).
 *
 *   states          DEVICE, const double[12][n_orbits]                       (read)
 *   out_states      DEVICE, double[12][n_orbits], may alias states            (written)
 *   out_invariants  DEVICE, double[12][n_orbits] or NULL: rows 0-5 = E, Jx, Jy, Jz, |S1hat|, |S2hat| of
 *                   the (normalised) input state, rows 6-11 = the same of the output state
 *   out_fli         DEVICE, double[n_orbits]; required iff shadow_eps != 0
 *
 * The call is asynchronous on params.cuda_stream: one kernel launch (preceded by one memset of the
 * work-queue scratch and, with params.regroup, by the key kernel and the sort), no host synchronisation, no host<->device copy.  All buffers are owned by the caller.  n_orbits = 0 or n_steps = 0 are valid
 * (n_steps = 0 copies the normalised state and evaluates the invariants).  Numerical failures of
 * single orbits are not errors: see mc_get_status.
 * Errors: MC_EINVAL (null/negative arguments, n_steps >= 2^31, unknown mode, non-finite step_h), MC_ECUDA. */
int mc_integrate(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                 int32_t correction_mode, double shadow_eps, double* out_states,
                 double* out_invariants, double* out_fli);

/* mc_integrate that also records the trajectory (the paper's phase portraits and spin-space
 * plots, are drawn from such samples): after every sample_interval-th step (k = interval,
 * 2 interval, ... <= n_steps) the state of every orbit (not of its shadow) is written to
 *   out_samples  DEVICE, double[n_steps / sample_interval][12][n_orbits]       (written)
 * A dropped orbit keeps reporting its frozen state.  sample_interval = 0 is mc_integrate.  The stores are
 * coalesced, streaming, and the only global traffic inside the step loop.
 * Errors: as mc_integrate; MC_EINVAL for a negative interval or a null out_samples with interval > 0. */
int mc_integrate_sampled(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                         int32_t correction_mode, double shadow_eps, double* out_states,
                         double* out_invariants, double* out_fli, int64_t sample_interval,
                         double* out_samples);

/* Checkpoint / resume: mc_integrate that also parks the COMPLETE state of the run -- orbit
 * and shadow, reference integrals E0, J0 of both, FLI accumulator, renormalisation counter,
 * status, step and Gauss-Newton counters -- in `carry`, a DEVICE buffer of mc_carry_bytes(n_orbits, shadow_eps != 0)
 * bytes owned by the caller, and with resume = 1 continues from it (`states` is then ignored and may be NULL).
 * n1 steps followed by a resumed call of n2 steps give, bit for bit, every output of one call of n1 + n2 steps
 * (same handle parameters, step_h, mode and shadow_eps; rows 0-5 of out_invariants, the initial integrals, are
 * written by the first call only; out_step and the work counter are cumulative).  The carry layout is private.
 * Errors: as mc_integrate; MC_EINVAL for a null carry or resume not in {0, 1}. */
int64_t mc_carry_bytes(int64_t n_orbits, int32_t with_shadow);
int mc_integrate_ex(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                    int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                    double* out_fli, void* carry, int32_t resume);

/* Same operation with HOST buffers (pageable or pinned): copies the inputs to device scratch owned by
 * the handle, runs mc_integrate, copies the outputs back and synchronises the stream before
 * returning.  out_status (int32[n_orbits]) and out_step (int64[n_orbits]) are optional host arrays. */
int mc_integrate_host(mc_handle* h, const double* states, int64_t n_orbits, double step_h,
                      int64_t n_steps, int32_t correction_mode, double shadow_eps, double* out_states,
                      double* out_invariants, double* out_fli, int32_t* out_status, int64_t* out_step);

/* mc_integrate for callers that must not allocate device memory.
 *
 * Why it exists.  A handle gets its device bookkeeping (work queue of the persistent kernel, per-orbit Gauss-Newton
 * counters, status arrays) from cudaMalloc, on first use and again whenever a batch is larger than any before.  That
 * is unusable for a program that has handed the whole GPU to its own memory pool (a later cudaMalloc by a library
 * just fails), for a loop with a latency budget (cudaMalloc / cudaFree stall all streams of the process), and
 * wherever the runtime refuses allocation outright, e.g. while a stream of the process is being captured.  This
 * entry point needs no handle and calls neither cudaMalloc nor cudaFree nor any library routine that allocates: its
 * bookkeeping lives in a fixed array compiled into libmc.so (256 bytes + 8 bytes x MC_STATIC_MAX_TRAJECTORIES, about
 * 256 KB).  Every GPU on which the library's code is loaded holds that array until the process exits, used or not.
 *
 * Same operation, arguments and kernel as mc_integrate, with these differences:
 *   params        what mc_create would be given, validated the same way on every call (nothing is created; per-orbit
 *                 parameter arrays must be valid for the duration of the launch); work is enqueued on
 *                 params->cuda_stream of params->device.  chunk_steps and regroup are ignored (one chunk, caller's
 *                 order: neither changes a result bit).  MC_TERM_RR is refused (MC_EINVAL): its extra outputs are
 *                 only reachable through a handle
 *   out_status    DEVICE int32[n_orbits] (mc_status) and
 *   out_step      DEVICE int64[n_orbits] (completed steps): REQUIRED here, written by the kernel directly -- what
 *                 mc_get_status would return
 *   limit         n_orbits x (shadow_eps != 0 ? 2 : 1) <= MC_STATIC_MAX_TRAJECTORIES, else MC_ELIMIT and nothing
 *                 is launched (mc_strerror(MC_ELIMIT) says so in words); larger batches need mc_integrate
 * Results are those of mc_integrate on the same inputs, bit for bit.
 *
 * First call on a device: looks up the device address of the fixed array and the SM count (once per device, cached)
 * and, like any first launch, makes the driver load the kernel.  Make that first call during start-up, before any
 * stream capture begins.  Later calls do: argument checks, one 256-byte cudaMemsetAsync, one kernel launch.
 *
 * Sharing.  All calls on one device use the same array, and it keeps what the previous call left there; the entry
 * point clears the part that must start at zero (the queue header) on the caller's stream.  Calls issued to the
 * same stream therefore just queue up.  Two calls of one process whose kernels can overlap on the GPU (issued to
 * different streams, from one host thread or several) would share one work queue: that is a data race with wrong
 * results, and it is the caller's job to order them (one stream, or an event between them).  Separate processes
 * each have their own copy of the array.
 * Errors: MC_EINVAL, MC_ELIMIT (both before any CUDA call), MC_EARCH, MC_ECUDA. */
#define MC_STATIC_MAX_TRAJECTORIES 32768
int mc_integrate_static(const mc_params* params, const double* states, int64_t n_orbits, double step_h,
                        int64_t n_steps, int32_t correction_mode, double shadow_eps, double* out_states,
                        double* out_invariants, double* out_fli, int32_t* out_status, int64_t* out_step);

/* Status of the orbits of the most recent mc_integrate on this handle, copied (stream-ordered) into
 * DEVICE arrays of the caller: out_status int32[n_orbits] (mc_status), out_step int64[n_orbits] =
 * number of completed steps.  Either pointer may be NULL. */
int mc_get_status(mc_handle* h, int32_t* out_status, int64_t* out_step);

/* Moving reference integrals of the most recent mc_integrate on a handle created with MC_TERM_RR, copied (stream-
 * ordered) into out_wg, DEVICE double[4][n_orbits]: E0 + W, J0x + Gx, J0y + Gy, J0z + Gz of every orbit at the end of
 * the run, W and G being the work and torque integrals of the radiation-reaction force (H(t) - W(t) and
 * J(t) - G(t) are constant along the exact flow, so rows 6-9 of out_invariants equal these to truncation error
 * without correction and to round-off with it; W = row 0 of this minus row 0 of out_invariants).  MC_EINVAL without
 * MC_TERM_RR. */
int mc_get_dissipation(mc_handle* h, double* out_wg);

/* Work done by the most recent mc_integrate on this handle: out_gn_steps, DEVICE int64[n_orbits] = number
 * of Gauss-Newton steps correction mode 3 took over all accepted steps of the orbit and its shadow
 * (0 for the other modes).  Stream-ordered copy.  bench.py derives the algorithmic flop count from it. */
int mc_get_work(mc_handle* h, int64_t* out_gn_steps);

/* What the warps of the most recent mc_integrate executed, summed over the launch, into HOST int64[2] (synchronises
 * the stream): [0] passes through the Gauss-Newton loop of mode 3 counted once per WARP (a warp repeats the loop while
 * any of its 32 lanes needs another step, so this exceeds the per-lane counts of mc_get_work divided by 32 by the
 * amount of divergence), [1] warp-steps (passes of a warp through the step loop).  bench.py uses both to convert the
 * SASS instruction mix into executed flop. */
int mc_get_warp_work(mc_handle* h, int64_t* out_host2);

/* Checked build only (libmc_checked.so, compiled with -DMC_CHECKED by paper_1802_00147_b200/build.py): the integration
 * kernel tests every index and pointer before the global access that uses it; *out_line (HOST) = 0 if no test of the most
 * recent mc_integrate failed, else the source line (csrc/mc_kernel.cuh) of the first one that did.  Synchronises the
 * stream.  The product library compiles the tests away and reports -1.  (compute-sanitizer is closed on this GPU pool;
 * the GPU tests run a representative set of launches through the checked library instead.) */
int mc_debug_check(mc_handle* h, int64_t* out_line);

/* Evaluate pieces of the model on the device with the handle's parameters (used by the parity tests
 * to compare the kernel's fused routines with the oracle one by one).  states: DEVICE double[12][n].
 *   what = 0: out[1][n]  = H                     (eq 1)
 *   what = 1: out[12][n] = dz/dt                 (eqs 6-9: dH/dp, -dH/dr, Omega_i x S_i_hat); with MC_TERM_RR
 *             out[16][n], rows 12-15 = dW/dt, dG/dt
 *   what = 2: out[6][n]  = E, Jx, Jy, Jz, |S1hat|, |S2hat|
 *   what = 3: out[12][n] = one step of the base integrator (params.integrator) of size step_h, no correction;
 *             with MC_TERM_RR out[16][n], rows 12-15 = W, G accumulated over the step (from zero); MC_EINVAL for the one
 *             combination that is not built (per_orbit = 1, MC_INTEG_RK5, MC_TERM_RR; see MC_TERM_RR)
 *   what = 4: out[12][n] = correction operator of mode `mode` applied to states, with references
 *             refs = DEVICE double[4][n] (E0, J0x, J0y, J0z); required for every mode (MC_EINVAL if NULL)
 * Asynchronous on the handle's stream. */
int mc_eval(mc_handle* h, int32_t what, const double* states, int64_t n, double step_h, int32_t mode,
            const double* refs, double* out);

/* Facts about the kernel the last mc_integrate launched (for bench.py / DESIGN.md evidence). */
typedef struct mc_launch_info {
  int32_t grid, block;          /* launch shape                                   */
  int32_t regs_per_thread;      /* cudaFuncAttributes.numRegs                     */
  int32_t local_bytes;          /* cudaFuncAttributes.localSizeBytes (spills)     */
  int32_t blocks_per_sm;        /* occupancy API result for that block size       */
  int32_t num_sms;
  int32_t smem_bytes;           /* dynamic shared memory per block                */
  int32_t variant;              /* bit0 per-orbit params, bit1 QM, bit2 per-orbit kq only, bit3 2.5PN, bits 4-5 mode, bit 8 RK5, bit 10 regrouped */
  int64_t trajectories;         /* threads doing work = n_orbits * (1 + shadow)   */
  int32_t chunk_steps;          /* steps per work item                             */
  int32_t n_chunks;             /* work items per 32-trajectory unit              */
} mc_launch_info;
int mc_last_launch_info(mc_handle* h, mc_launch_info* out);

int mc_destroy(mc_handle* h);

/* Static string for an mc_error; for MC_ECUDA the text of the last CUDA error seen by this thread. */
const char* mc_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* MC_H_ */
