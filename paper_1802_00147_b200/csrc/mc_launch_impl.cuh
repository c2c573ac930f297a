// mc_launch_impl.cuh -- included by mc_kernel_mode<N>.cu with MC_MODE defined.
#pragma once
#include <type_traits>

#include "mc_kernel.cuh"
#include "mc_launch.h"

namespace mc {

// Resident 128-thread blocks per SM the register allocator must allow.  With constant-bank parameters (uniform, or
// uniform + per-orbit kappa in four registers) the RK4 kernels fit 3 blocks (<= 168 registers) without spills, with
// or without the quadrupole-monopole term.  Fully per-orbit parameters (45 constants in shared memory) and the
// six-stage RK5 need <= 255 registers (2 blocks).  ptxas -v: 0 spill bytes for every instantiation (build() raises
// otherwise).
#ifndef MC_MINB_UNIFORM
#define MC_MINB_UNIFORM 3
#endif
#ifndef MC_MINB_PER_ORBIT
#define MC_MINB_PER_ORBIT 2
#endif

template <int PARAMS, bool QM, int MODE, int INTEG, bool RR>
static cudaError_t launch(const McConsts& uc, const IntegrateArgs& A, int num_sms, bool do_launch, cudaStream_t stream,
                          KernelInfo* info) {
  auto kern = integrate_kernel<PARAMS, QM, MODE, INTEG, RR, ((PARAMS == PARAMS_PER_ORBIT || INTEG == 1 || RR) ? MC_MINB_PER_ORBIT : MC_MINB_UNIFORM)>;
  const size_t smem = PARAMS == PARAMS_PER_ORBIT ? sizeof(double) * MC_NCONST * kBlock : 0;
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, kern);
  if (e != cudaSuccess) return e;
  int bps = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kern, kBlock, smem);
  if (e != cudaSuccess) return e;
  if (bps < 1) return cudaErrorLaunchOutOfResources;
  const int64_t need = (A.n_units * 32 + kBlock - 1) / kBlock;           // blocks if every unit had its own warp
  const int64_t cap = (int64_t)num_sms * bps;                              // blocks resident at once
  const int grid = (int)(need < cap ? need : cap);
  if (info) {
    info->regs = fa.numRegs;
    info->local_bytes = (int)fa.localSizeBytes;
    info->block = kBlock;
    info->smem = smem;
    info->blocks_per_sm = bps;
    info->grid = grid;
  }
  if (do_launch && grid > 0) kern<<<grid, kBlock, smem, stream>>>(uc, A);
  return cudaGetLastError();
}

// params: 0 uniform, 1 per orbit, 2 per-orbit kappa only (meaningful with the QM term; without it kappa is unused
// and the uniform kernel runs); rr: 2.5PN radiation reaction (16-component trajectories)
template <int MODE, int INTEG, bool RR>
static LaunchFn pick3(int params, bool qm) {
  if (params == PARAMS_PER_ORBIT) {
    // 45 per-orbit constants + six RK5 stages + the 16-component trajectory do not fit 255 registers: that one
    // combination is not built (mc_integrate returns MC_EINVAL; include/mc.h, MC_TERM_RR)
    if constexpr (INTEG == 1 && RR) return nullptr;
    else return qm ? launch<PARAMS_PER_ORBIT, true, MODE, INTEG, RR> : launch<PARAMS_PER_ORBIT, false, MODE, INTEG, RR>;
  }
  if (params == PARAMS_KAPPA && qm) return launch<PARAMS_KAPPA, true, MODE, INTEG, RR>;
  return qm ? launch<PARAMS_UNIFORM, true, MODE, INTEG, RR> : launch<PARAMS_UNIFORM, false, MODE, INTEG, RR>;
}

template <int MODE>
static LaunchFn pick(int params, bool qm, int integrator, bool rr) {
  if (rr) return integrator == 1 ? pick3<MODE, 1, true>(params, qm) : pick3<MODE, 0, true>(params, qm);
  return integrator == 1 ? pick3<MODE, 1, false>(params, qm) : pick3<MODE, 0, false>(params, qm);
}

}  // namespace mc
