// mc_kernel.cuh -- the integration kernel: one thread per trajectory, whole state in registers inside
// the step loop; with a shadow, lanes (2k, 2k+1) of a warp hold orbit k's main and shadow trajectory and
// meet through warp shuffles (status every step, distance every renorm_interval steps).
//
// Scheduling: the grid is persistent (as many blocks as are resident at once) and
// every WARP pulls work items from a global queue.  An item is (chunk c, unit u): unit u = 32 consecutive
// trajectories, chunk c = steps [c*chunk_len, (c+1)*chunk_len).  Items are numbered chunk-major, so unit
// u's chunk c+1 is handed out n_units items after its chunk c; between chunks the trajectory state
// (17 doubles + 20 bytes) rests in an L2-resident carry buffer and a per-unit flag publishes it.  When
// everything is resident at once there is one chunk and no carry traffic.  Otherwise the chunks remove
// the partial last wave: all SMs stay busy until the last chunk.
// Global memory is touched at launch, at chunk boundaries and at the end only, always coalesced SoA.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "mc_correct.cuh"

namespace mc {

struct IntegrateArgs {
  const double* states;      // [12][n]
  double* out_states;        // [12][n]
  double* out_inv;           // [12][n] or null
  double* out_fli;           // [n] or null
  int32_t* out_status;       // [n]
  int64_t* out_step;         // [n]
  int64_t* out_gn;           // [n] Gauss-Newton steps of mode 3 over accepted steps, orbit + shadow
  const double* beta; const double* chi1; const double* chi2; const double* kq1; const double* kq2;  // per-orbit mode
  const int32_t* perm;       // [n] or null: the orbit that slot s of the launch integrates (mc_params.regroup; scheduling only)
  int64_t n;                 // orbits
  int64_t n_steps;
  double h;
  StepWeights hw;            // h times the tableau coefficients (step_weights(h)): constant-bank operands of the stage sums
  double shadow_eps;         // 0: no shadow
  double r_merge2, r_escape2;
  double newton_tol;
  uint32_t terms;
  int32_t renorm_interval;
  int32_t newton_iters;
  int32_t integrator;         // 0 RK4, 1 RK5 (mc_eval only; integrate_kernel is instantiated per integrator)
  double* samples;            // [n_steps / sample_interval][12][n] or null: orbit states after steps interval, 2 interval, ...
  int32_t sample_interval;
  // scheduling
  unsigned long long* queue;  // [0] = next item; [1] += Gauss-Newton passes of the warps; [2] += warp-steps executed (mc_get_warp_work)
  int32_t* done;              // [n_units] chunks completed per unit
  double* carry_d;            // [17][n_traj_padded]: y[12], E0, J0[3] (MC_TERM_RR: E0 + W, J0 + G), acc
  double* out_diss;           // [4][n]: E0 + W, J0 + G of the orbit at the end (MC_TERM_RR), handle-owned
  int32_t* carry_i;           // [2][n_traj_padded]: status | flag << 8 | frozen << 31, until_renorm
  unsigned long long* carry_g;  // [2][n_traj_padded]: Gauss-Newton steps, completed steps (64-bit: they accumulate over resumed calls)
  int64_t n_units;            // ceil(trajectories / 32)
  int64_t n_items;            // n_units * n_chunks
  int32_t chunk_len;          // steps per chunk (>= 1)
  int32_t n_chunks;
  int32_t resume;             // 1: chunk 0 starts from the carry buffer instead of `states` (mc_integrate_ex)
  int32_t save_final;         // 1: the last chunk also parks its state in the carry buffer (mc_integrate_ex)
  unsigned long long wait_budget_ns;  // a warp waiting longer than this for its unit's previous chunk traps (mc_params.wait_budget_s)
};

// Checked build (-DMC_CHECKED, libmc_checked.so; compute-sanitizer is closed on this GPU pool): every index and pointer
// the kernel is about to use for a global access is tested first; the source line of the first failed test lands in
// queue[3] (mc_debug_check).  The product build compiles the tests away.
#ifdef MC_CHECKED
#define MC_CHK(cond) do { if (!(cond)) atomicCAS(A.queue + 3, 0ULL, (unsigned long long)__LINE__); } while (0)
#else
#define MC_CHK(cond) do { } while (0)
#endif

#ifndef MC_BLOCK
#define MC_BLOCK 128
#endif
constexpr int kBlock = MC_BLOCK;

template <bool QM, class C>
__device__ __forceinline__ void six_integrals(const C& c, const double* z, double* out6) {
  out6[0] = hamiltonian<QM>(c, z);
  total_J(c, z, out6 + 1);
  out6[4] = sqrt(dot3(z + 6, z + 6));
  out6[5] = sqrt(dot3(z + 9, z + 9));
}

// Register budget: either "MINB resident blocks" (__launch_bounds__) or, with MC_MAXNREG defined, an
// explicit per-thread cap (__maxnreg__; the two qualifiers exclude each other).
#ifdef MC_MAXNREG
#define MC_KERNEL_BOUNDS(MINB) __maxnreg__(MC_MAXNREG)
#else
#define MC_KERNEL_BOUNDS(MINB) __launch_bounds__(kBlock, MINB)
#endif

// PARAMS: 0 uniform parameters (constant bank), 1 every parameter per orbit (derived constants in shared memory),
// 2 uniform beta, chi with per-orbit quadrupole coefficients (KappaConsts; instantiated with QM only).
enum { PARAMS_UNIFORM = 0, PARAMS_PER_ORBIT = 1, PARAMS_KAPPA = 2 };

template <int PARAMS, class CP>
__device__ __forceinline__ CP make_consts(const McConsts& uc, const IntegrateArgs& A, int64_t orbit, double* smem) {
  if constexpr (PARAMS == PARAMS_PER_ORBIT) {
    mc_derive_consts(A.beta[orbit], A.chi1[orbit], A.chi2[orbit], A.kq1[orbit], A.kq2[orbit], A.terms,
                     smem + threadIdx.x, kBlock);
    return SharedConsts{smem + threadIdx.x, kBlock};
  } else if constexpr (PARAMS == PARAMS_KAPPA) {
    const double k1 = A.kq1[orbit], k2 = A.kq2[orbit];
    return KappaConsts{uc, k1 * uc.v[K_Q1], k2 * uc.v[K_Q2], k1 * uc.v[K_3M11], k2 * uc.v[K_3M22]};
  } else {
    return UniformConsts{uc};
  }
}
template <int PARAMS> struct ConstsOf { typedef UniformConsts type; };
template <> struct ConstsOf<PARAMS_PER_ORBIT> { typedef SharedConsts type; };
template <> struct ConstsOf<PARAMS_KAPPA> { typedef KappaConsts type; };

// RR: 2.5PN radiation reaction (MC_TERM_RR): the correction targets E0 + W, J0 + G, W and G being the work and torque
// integrals of the force (R21).  W and G enter nowhere else, so the trajectory carries the
// MOVING REFERENCES themselves as components 12-15 through the RK step (initial values E0, J0, rates dW/dt, dG/dt)
// and the separate reference registers R are not used.
template <int PARAMS, bool QM, int MODE, int INTEG, bool RR, int MINB>
__global__ void MC_KERNEL_BOUNDS(MINB)
integrate_kernel(const __grid_constant__ McConsts uc, const __grid_constant__ IntegrateArgs A) {
  constexpr int NS = RR ? 16 : 12;
  extern __shared__ double smem[];   // PARAMS_PER_ORBIT: [MC_NCONST][kBlock]
  const bool shadow = A.shadow_eps != 0.0;
  const int lane = threadIdx.x & 31;
  const int64_t tp = A.n_units * 32;   // padded trajectory count = stride of the carry arrays
  const double d0 = fabs(A.shadow_eps);
  const int n_steps = (int)A.n_steps;  // < 2^31 (mc_integrate checks)

#pragma unroll 1
  for (;;) {
    unsigned long long item = 0;
    if (lane == 0) item = atomicAdd(A.queue, 1ULL);
    item = __shfl_sync(0xffffffffu, item, 0);
    if (item >= (unsigned long long)A.n_items) break;
    const int chunk = (int)(item / (unsigned long long)A.n_units);
    const int64_t unit = (int64_t)(item % (unsigned long long)A.n_units);
    const int64_t t = unit * 32 + lane;
    const int64_t orbit_raw = shadow ? (t >> 1) : t;
    const bool role_shadow = shadow && (t & 1);
    const bool active = orbit_raw < A.n;
    const int64_t slot = active ? orbit_raw : (A.n - 1);    // idle lanes shadow-compute a valid orbit, never store
    MC_CHK(slot >= 0 && slot < A.n);
    const int64_t orbit = A.perm ? (int64_t)A.perm[slot] : slot;   // which orbit this slot holds: an index mapping only
    MC_CHK(unit >= 0 && unit < A.n_units && chunk >= 0 && chunk < A.n_chunks);
    MC_CHK(t >= 0 && t < tp && orbit >= 0 && orbit < A.n);
    MC_CHK(PARAMS == PARAMS_UNIFORM || (A.kq1 != nullptr && A.kq2 != nullptr));
    MC_CHK(PARAMS != PARAMS_PER_ORBIT || (A.beta != nullptr && A.chi1 != nullptr && A.chi2 != nullptr));

    using CP = typename ConstsOf<PARAMS>::type;
    const CP c = make_consts<PARAMS, CP>(uc, A, orbit, smem);

    double y[NS];
    Refs R;
    int status = ST_OK, flag = 0;
    bool frozen = false;
    // accepted steps and Gauss-Newton steps of THIS work item (chunk): 32-bit in the loop; the 64-bit totals of
    // earlier chunks / earlier calls stay in the carry buffer and are added when the item is parked or stored
    int steps = 0;
    unsigned gn_chunk = 0;
    unsigned gn_warp = 0, warp_steps = 0;  // passes of this WARP through the Gauss-Newton loop / the step loop (work accounting)
    double acc = 0.0;
    int until_renorm = A.renorm_interval;

    if (chunk == 0 && !A.resume) {
      // prologue: coalesced SoA load, eq (10) on the input, reference integrals
      MC_CHK(A.states != nullptr);
#pragma unroll
      for (int i = 0; i < 12; ++i) y[i] = A.states[(int64_t)i * A.n + orbit];
      if (MODE >= 1) { normalise3(y + 6); normalise3(y + 9); }
      if (!role_shadow && active && A.out_inv) {   // rows 0-5: the main trajectory before the offset
        double inv0[6];
        six_integrals<QM>(c, y, inv0);
#pragma unroll
        for (int i = 0; i < 6; ++i) A.out_inv[(int64_t)i * A.n + orbit] = inv0[i];
      }
      if (role_shadow) y[0] += A.shadow_eps;
      references<QM>(c, y, R);
      if constexpr (RR) { y[12] = R.E0; y[13] = R.J0[0]; y[14] = R.J0[1]; y[15] = R.J0[2]; }
    } else {
      // wait until this unit's previous chunk is published, then reload the carried state.  The holder of
      // that chunk got it earlier from the same queue, so it is running -- PROVIDED the whole grid is resident at
      // once, which the launcher guarantees by sizing the grid with the occupancy API (mc_launch_impl.cuh); under
      // MPS or any other co-tenant that takes SM resources between the query and the launch that no longer holds,
      // hence the budget: a wait longer than mc_params.wait_budget_s traps (the launch fails) instead of hanging.
      if (chunk > 0 && lane == 0) {
        unsigned long long t0 = 0;
        while (*(volatile int32_t*)(A.done + unit) < chunk) {
          __nanosleep(200);
          unsigned long long now;
          asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
          if (t0 == 0) t0 = now;
          else if (now - t0 > A.wait_budget_ns) __trap();         // fail loudly instead of hanging
        }
      }
      // acquire, mirroring the publish side below: the lane that observed the flag issues the fence, the barrier then
      // orders every lane's ld.cg after it (a resumed chunk 0 has no flag to observe: the previous launch has ended)
      if (lane == 0) __threadfence();
      __syncwarp();
      MC_CHK(A.carry_d != nullptr && A.carry_i != nullptr && A.carry_g != nullptr && A.done != nullptr);
#pragma unroll
      for (int i = 0; i < 12; ++i) y[i] = __ldcg(A.carry_d + (int64_t)i * tp + t);   // L2 only: L1 may be stale
      R.E0 = __ldcg(A.carry_d + 12 * tp + t);
#pragma unroll
      for (int i = 0; i < 3; ++i) R.J0[i] = __ldcg(A.carry_d + (int64_t)(13 + i) * tp + t);
      acc = __ldcg(A.carry_d + 16 * tp + t);
      if constexpr (RR) { y[12] = R.E0; y[13] = R.J0[0]; y[14] = R.J0[1]; y[15] = R.J0[2]; }
      const int packed = __ldcg(A.carry_i + t);
      status = packed & 0xff;
      flag = (packed >> 8) & ST_NEWTON_FLAG;   // bit 16 -> 256
      frozen = packed < 0;
      until_renorm = __ldcg(A.carry_i + tp + t);
    }

    // steps until the next sample; a countdown instead of a modulo in the step loop
    int until_sample = (A.samples != nullptr) ? A.sample_interval - (int)(((long long)chunk * A.chunk_len) % A.sample_interval) : 0x7fffffff;
    const int k_end = min(n_steps, (chunk + 1 == A.n_chunks) ? n_steps : (chunk + 1) * A.chunk_len);
#pragma unroll 1
    for (int k = chunk * A.chunk_len; k < k_end; ++k) {
      if (__all_sync(0xffffffffu, frozen)) {
        if (A.samples != nullptr && !role_shadow && active) {      // whole warp dropped: remaining samples of this chunk
          for (int kk = k; kk < k_end; ++kk)
            if ((kk + 1) % A.sample_interval == 0) {
              MC_CHK((kk + 1) / A.sample_interval >= 1 && (kk + 1) / A.sample_interval <= A.n_steps / A.sample_interval);
              double* dst = A.samples + ((int64_t)((kk + 1) / A.sample_interval - 1) * 12) * A.n + orbit;
#pragma unroll
              for (int i = 0; i < 12; ++i) __stcs(dst + (int64_t)i * A.n, y[i]);
            }
        }
        break;
      }
      ++warp_steps;
      double z[NS];
      base_step<INTEG, QM, RR>(c, y, A.hw, z);
      int gn, gnw;
      bool ok;
      if constexpr (RR) {   // the manifold has moved by the work and torque of the step (integral invariant relation)
        Refs Rm;
        Rm.E0 = z[12]; Rm.J0[0] = z[13]; Rm.J0[1] = z[14]; Rm.J0[2] = z[15];
        ok = correct<MODE, QM>(c, z, Rm, A.newton_iters, A.newton_tol, gn, gnw);
      } else {
        ok = correct<MODE, QM>(c, z, R, A.newton_iters, A.newton_tol, gn, gnw);
      }
      gn_warp += (unsigned)gnw;
      if (MODE == 2 && !ok && !role_shadow && !frozen) flag = ST_NEWTON_FLAG;
      // status of the completed step (R13): non-finite anywhere in the pair, else |r| of the main
      int code = ST_OK;
      if (!finite12(z)) code = ST_NONFINITE;
      else if (!role_shadow) code = radius_status(z, A.r_merge2, A.r_escape2);
      if (shadow) {
        const int other = __shfl_xor_sync(0xffffffffu, code, 1);
        code = (code == ST_NONFINITE || other == ST_NONFINITE) ? ST_NONFINITE : (role_shadow ? other : code);
      }
      if (!frozen) {
        if (code == ST_OK) {
#pragma unroll
          for (int i = 0; i < NS; ++i) y[i] = z[i];
          ++steps;
          gn_chunk += (unsigned)gn;
        } else {
          frozen = true;
          status = code;
        }
      }
      if (--until_sample == 0) {
        // sampled output: the orbit's current state, its frozen state once it has been dropped
        until_sample = A.sample_interval;
        if (!role_shadow && active) {
          MC_CHK(A.samples != nullptr && (k + 1) / A.sample_interval >= 1 && (k + 1) / A.sample_interval <= A.n_steps / A.sample_interval);
          double* dst = A.samples + ((int64_t)((k + 1) / A.sample_interval - 1) * 12) * A.n + orbit;
#pragma unroll
          for (int i = 0; i < 12; ++i) __stcs(dst + (int64_t)i * A.n, y[i]);
        }
      }
      if (shadow && --until_renorm == 0) {
        until_renorm = A.renorm_interval;
        // shadow lane pulls the main state; d = |z' - z| over all 12 components (R10, R12)
        double ym[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) ym[i] = __shfl_xor_sync(0xffffffffu, y[i], 1);
        int bad = 0;
        if (role_shadow && !frozen) {
          // distance, FLI term, pull-back, eq (10), re-referenced integrals (R11): mc_correct.cuh
          if (!renormalise_shadow<MODE, QM>(c, y, ym, d0, acc, R)) bad = 1;
          else if constexpr (RR) { y[12] = R.E0; y[13] = R.J0[0]; y[14] = R.J0[1]; y[15] = R.J0[2]; }   // W, G restart with them
        }
        bad |= __shfl_xor_sync(0xffffffffu, bad, 1);
        if (bad && !frozen) { frozen = true; status = ST_NONFINITE; }
      }
    }

    if (lane == 0) {   // what the pipe executed, per launch (mc_get_warp_work)
      atomicAdd(A.queue + 1, (unsigned long long)gn_warp);
      atomicAdd(A.queue + 2, (unsigned long long)warp_steps);
    }
    const bool last = chunk + 1 == A.n_chunks;
    const bool carried = chunk > 0 || A.resume;
    unsigned long long gn_total = gn_chunk;
    long long steps_total = steps;
    if (carried) {
      gn_total += __ldcg(A.carry_g + t);
      steps_total += (long long)__ldcg(A.carry_g + tp + t);
    }
    if (!last || A.save_final) {
      // park the state in the carry buffer (and publish the chunk unless it is the last)
      MC_CHK(A.carry_d != nullptr && A.carry_i != nullptr && A.carry_g != nullptr && A.done != nullptr);
#pragma unroll
      for (int i = 0; i < 12; ++i) __stcg(A.carry_d + (int64_t)i * tp + t, y[i]);
      if constexpr (RR) { R.E0 = y[12]; R.J0[0] = y[13]; R.J0[1] = y[14]; R.J0[2] = y[15]; }
      __stcg(A.carry_d + 12 * tp + t, R.E0);
#pragma unroll
      for (int i = 0; i < 3; ++i) __stcg(A.carry_d + (int64_t)(13 + i) * tp + t, R.J0[i]);
      __stcg(A.carry_d + 16 * tp + t, acc);
      __stcg(A.carry_i + t, (status & 0xff) | (flag << 8) | (frozen ? (int)0x80000000 : 0));
      __stcg(A.carry_i + tp + t, until_renorm);
      __stcg(A.carry_g + t, gn_total);
      __stcg(A.carry_g + tp + t, (unsigned long long)steps_total);
      if (!last) {
        // publish: the barrier collects every lane's st.cg, then the lane that writes the flag issues the release
        // fence (cumulativity: it covers the stores it observed through the barrier) and the flag store
        __syncwarp();
        if (lane == 0) { __threadfence(); atomicExch(A.done + unit, chunk + 1); }
        continue;
      }
    }

    // epilogue: FLI from the final separation, invariants, coalesced SoA stores
    MC_CHK(A.out_states != nullptr && A.out_status != nullptr && A.out_step != nullptr && A.out_gn != nullptr);
    MC_CHK(!shadow || A.out_fli != nullptr);
    MC_CHK(!RR || A.out_diss != nullptr);
    if (shadow) gn_total += __shfl_xor_sync(0xffffffffu, gn_total, 1);
    if (shadow) {
      double ym[12];
#pragma unroll
      for (int i = 0; i < 12; ++i) ym[i] = __shfl_xor_sync(0xffffffffu, y[i], 1);
      if (role_shadow && active) {
        double d2 = 0.0;
#pragma unroll
        for (int i = 0; i < 12; ++i) { const double e = y[i] - ym[i]; d2 = fma(e, e, d2); }
        A.out_fli[orbit] = acc + log10(sqrt(d2) / d0);
      }
    }
    if (!role_shadow && active) {
#pragma unroll
      for (int i = 0; i < 12; ++i) A.out_states[(int64_t)i * A.n + orbit] = y[i];
      if (A.out_inv) {
        double inv1[6];
        six_integrals<QM>(c, y, inv1);
#pragma unroll
        for (int i = 0; i < 6; ++i) A.out_inv[(int64_t)(6 + i) * A.n + orbit] = inv1[i];
      }
      if constexpr (RR) {
#pragma unroll
        for (int i = 0; i < 4; ++i) A.out_diss[(int64_t)i * A.n + orbit] = y[12 + i];
      }
      A.out_status[orbit] = status | flag;
      A.out_step[orbit] = steps_total;
      A.out_gn[orbit] = (int64_t)gn_total;
    }
  }
}

}  // namespace mc
