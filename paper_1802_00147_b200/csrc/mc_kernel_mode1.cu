// integrate_kernel instantiations for correction mode 1 (include/mc.h: mc_correction).
#include "mc_launch_impl.cuh"
namespace mc {
LaunchFn launcher_mode1(int params, bool qm, int integrator, bool rr) { return pick<1>(params, qm, integrator, rr); }
}  // namespace mc
