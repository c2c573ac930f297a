// integrate_kernel instantiations for correction mode 0 (include/mc.h: mc_correction).
#include "mc_launch_impl.cuh"
namespace mc {
LaunchFn launcher_mode0(int params, bool qm, int integrator, bool rr) { return pick<0>(params, qm, integrator, rr); }
}  // namespace mc
