// integrate_kernel instantiations for correction mode 2 (include/mc.h: mc_correction).
#include "mc_launch_impl.cuh"
namespace mc {
LaunchFn launcher_mode2(int params, bool qm, int integrator, bool rr) { return pick<2>(params, qm, integrator, rr); }
}  // namespace mc
