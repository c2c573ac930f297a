// mc_launch.h -- host-side table of the integrate_kernel instantiations (one .cu per correction mode
// so the heavy kernels compile in parallel).
#pragma once
#include <cuda_runtime.h>

#include "mc_consts.h"

namespace mc {
struct IntegrateArgs;
struct KernelInfo { int regs, local_bytes, blocks_per_sm, block, grid; size_t smem; };
// query: fills KernelInfo (occupancy, registers) without launching.  launch: starts min(blocks needed,
// resident capacity) persistent blocks.
typedef cudaError_t (*LaunchFn)(const McConsts&, const IntegrateArgs&, int num_sms, bool do_launch, cudaStream_t, KernelInfo*);
LaunchFn launcher_mode0(int params, bool qm, int integrator, bool rr);
LaunchFn launcher_mode1(int params, bool qm, int integrator, bool rr);
LaunchFn launcher_mode2(int params, bool qm, int integrator, bool rr);
LaunchFn launcher_mode3(int params, bool qm, int integrator, bool rr);
// mc_api.cu: stores the text mc_strerror(MC_ECUDA) returns on this thread; returns MC_ECUDA (for mc_static.cu)
int record_cuda_failure(cudaError_t e);
}  // namespace mc
