// mc_kernel.cuh -- the integration kernel: one thread per trajectory, whole state in registers for
// all n_steps; with a shadow, lanes (2k, 2k+1) of a warp hold orbit k's main and shadow trajectory and
// meet through warp shuffles (status every step, distance every renorm_interval steps).
// Global memory is touched at launch (coalesced SoA loads) and at the end (coalesced SoA stores) only.
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
  int64_t n;                 // orbits
  int64_t n_steps;
  double h;
  double shadow_eps;         // 0: no shadow
  double r_merge2, r_escape2;
  double newton_tol;
  uint32_t terms;
  int32_t renorm_interval;
  int32_t newton_iters;
};

enum { ST_OK = 0, ST_MERGED = 1, ST_UNBOUND = 2, ST_NONFINITE = 3, ST_NEWTON_FLAG = 256 };

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

template <bool PER_ORBIT, bool QM, int MODE, int MINB>
__global__ void MC_KERNEL_BOUNDS(MINB)
integrate_kernel(const __grid_constant__ McConsts uc, const __grid_constant__ IntegrateArgs A) {
  extern __shared__ double smem[];   // PER_ORBIT: [MC_NCONST][kBlock]
  const bool shadow = A.shadow_eps != 0.0;
  const int64_t t = (int64_t)blockIdx.x * kBlock + threadIdx.x;
  const int64_t orbit_raw = shadow ? (t >> 1) : t;
  const bool role_shadow = shadow && (t & 1);
  const bool active = orbit_raw < A.n;
  const int64_t orbit = active ? orbit_raw : (A.n - 1);   // idle lanes shadow-compute a valid orbit, never store

  using CP = typename std::conditional<PER_ORBIT, SharedConsts, UniformConsts>::type;
  CP c = [&]() {
    if constexpr (PER_ORBIT) {
      mc_derive_consts(A.beta[orbit], A.chi1[orbit], A.chi2[orbit], A.kq1[orbit], A.kq2[orbit], A.terms,
                       smem + threadIdx.x, kBlock);
      return SharedConsts{smem + threadIdx.x, kBlock};
    } else {
      return UniformConsts{uc};
    }
  }();

  double y[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) y[i] = A.states[(int64_t)i * A.n + orbit];
  if (MODE >= 1) { normalise3(y + 6); normalise3(y + 9); }
  if (!role_shadow && active && A.out_inv) {   // rows 0-5: the main trajectory before the offset; stored now so
    double inv0[6];                            // that nothing of it stays in registers during the step loop
    six_integrals<QM>(c, y, inv0);
#pragma unroll
    for (int i = 0; i < 6; ++i) A.out_inv[(int64_t)i * A.n + orbit] = inv0[i];
  }
  const double d0 = fabs(A.shadow_eps);
  if (role_shadow) y[0] += A.shadow_eps;
  Refs R;
  references<QM>(c, y, R);

  int status = ST_OK, flag = 0;
  bool frozen = false;
  int steps = 0;            // n_steps < 2^31 (mc_integrate checks)
  unsigned long long gn_total = 0;
  double acc = 0.0;
  int until_renorm = A.renorm_interval;

  const int n_steps = (int)A.n_steps;
#pragma unroll 1
  for (int k = 0; k < n_steps; ++k) {
    double z[12];
    rk4_step<QM>(c, y, A.h, z);
    int gn;
    const bool ok = correct<MODE, QM>(c, z, R, A.newton_iters, A.newton_tol, gn);
    if (MODE == 2 && !ok && !role_shadow && !frozen) flag = ST_NEWTON_FLAG;
    // status of the completed step (R13): non-finite anywhere in the pair, else |r| of the main
    int code = ST_OK;
    if (!finite12(z)) code = ST_NONFINITE;
    else if (!role_shadow) {
      const double r2 = dot3(z, z);
      code = (r2 < A.r_merge2) ? ST_MERGED : ((r2 > A.r_escape2) ? ST_UNBOUND : ST_OK);
    }
    if (shadow) {
      const int other = __shfl_xor_sync(0xffffffffu, code, 1);
      code = (code == ST_NONFINITE || other == ST_NONFINITE) ? ST_NONFINITE : (role_shadow ? other : code);
    }
    if (!frozen) {
      if (code == ST_OK) {
#pragma unroll
        for (int i = 0; i < 12; ++i) y[i] = z[i];
        ++steps;
        gn_total += (unsigned)gn;
      } else {
        frozen = true;
        status = code;
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
        double d2 = 0.0;
#pragma unroll
        for (int i = 0; i < 12; ++i) { const double e = y[i] - ym[i]; d2 = fma(e, e, d2); }
        const double d = sqrt(d2);
        if (!(d > 0.0) || !(d < 1.0e300)) {
          bad = 1;
        } else {
          acc += log10(d / d0);
          const double s = d0 / d;
#pragma unroll
          for (int i = 0; i < 12; ++i) y[i] = fma(s, y[i] - ym[i], ym[i]);
          if (MODE >= 1) { normalise3(y + 6); normalise3(y + 9); }
          references<QM>(c, y, R);   // the shadow obeys its own, re-referenced integrals (R11)
        }
      }
      bad |= __shfl_xor_sync(0xffffffffu, bad, 1);
      if (bad && !frozen) { frozen = true; status = ST_NONFINITE; }
    }
    if (__all_sync(0xffffffffu, frozen)) break;
  }

  // epilogue: FLI from the final separation, invariants, coalesced SoA stores
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
    A.out_status[orbit] = status | flag;
    A.out_step[orbit] = steps;
    A.out_gn[orbit] = (int64_t)gn_total;
  }
}

}  // namespace mc
