// mc_launch_impl.cuh -- included by mc_kernel_mode<N>.cu with MC_MODE defined.
#pragma once
#include <type_traits>

#include "mc_kernel.cuh"
#include "mc_launch.h"

namespace mc {

// Resident 128-thread blocks per SM the register allocator must allow.  Uniform parameters are
// constant-bank operands, so 3 blocks (<= 168 registers) fit without spills; per-orbit parameters, the
// quadrupole-monopole term and the six-stage RK5 need <= 255 registers (2 blocks; within 6 % of the 3-block
// speed, profiles/r01_config_sweep.md).  ptxas -v: 0 spill bytes for all 32 instantiations (checked by build()).
#ifndef MC_MINB_UNIFORM
#define MC_MINB_UNIFORM 3
#endif
#ifndef MC_MINB_PER_ORBIT
#define MC_MINB_PER_ORBIT 2
#endif

template <bool PER_ORBIT, bool QM, int MODE, int INTEG>
static cudaError_t launch(const McConsts& uc, const IntegrateArgs& A, int num_sms, bool do_launch, cudaStream_t stream,
                          KernelInfo* info) {
  auto kern = integrate_kernel<PER_ORBIT, QM, MODE, INTEG, ((PER_ORBIT || QM || INTEG == 1) ? MC_MINB_PER_ORBIT : MC_MINB_UNIFORM)>;
  const size_t smem = PER_ORBIT ? sizeof(double) * MC_NCONST * kBlock : 0;
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

template <int MODE, int INTEG>
static LaunchFn pick2(bool per_orbit, bool qm) {
  if (per_orbit) return qm ? launch<true, true, MODE, INTEG> : launch<true, false, MODE, INTEG>;
  return qm ? launch<false, true, MODE, INTEG> : launch<false, false, MODE, INTEG>;
}

template <int MODE>
static LaunchFn pick(bool per_orbit, bool qm, int integrator) {
  return integrator == 1 ? pick2<MODE, 1>(per_orbit, qm) : pick2<MODE, 0>(per_orbit, qm);
}

}  // namespace mc
