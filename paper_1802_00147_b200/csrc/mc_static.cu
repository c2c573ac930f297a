// mc_static.cu -- mc_integrate_static (include/mc.h): the integration kernel for callers that may not allocate.
//
// Who this is for.  mc_integrate keeps its bookkeeping (the warps' work queue, the per-orbit Gauss-Newton counters,
// the status arrays) in device buffers that the handle obtains from cudaMalloc the first time they are needed and
// whenever a batch is larger than the last one.  Some programs cannot have a library do that on their behalf:
//   * a host application or framework that takes all of the GPU's memory for its own pool at start-up, so that a
//     later cudaMalloc from anybody else simply fails;
//   * a service loop with a latency budget: cudaMalloc and cudaFree are synchronising, slow calls that stall every
//     stream of the process, and a batch that happens to be larger than the previous one would hit them mid-flight;
//   * code running where the CUDA runtime forbids allocation altogether, for instance while one of the process's
//     streams is being captured, when cudaMalloc is an error that also invalidates the capture.
// For them the bookkeeping lives in the fixed array below, which is part of the library image: the driver places it
// in device memory when the library's module is loaded on a GPU and releases it when the process ends, so every GPU
// that runs this library holds these 256 KB whether or not the entry point is ever called.  The price is a hard
// upper limit on the batch (MC_STATIC_MAX_TRAJECTORIES) and that all calls on a device share the one array.
//
// The kernel is the same integrate_kernel every other entry point launches, always as ONE chunk (every unit of a batch
// this small is resident at once, so there is nothing to balance and no carry buffer is needed).
#include <cuda_runtime.h>

#include <cmath>
#include <cstring>
#include <mutex>

#include "../../include/mc.h"
#include "mc_kernel.cuh"
#include "mc_launch.h"

namespace {

// Layout of the fixed scratch: [0, 256) the work queue header (four 64-bit words: next item, two work counters,
// the checked build's line slot), then one 64-bit Gauss-Newton counter per orbit.
constexpr size_t kQueueBytes = 256;
constexpr size_t kScratchBytes = kQueueBytes + sizeof(int64_t) * (size_t)MC_STATIC_MAX_TRAJECTORIES;

// In HOST code this name is only a handle for the runtime's symbol table, NOT an address the GPU understands: the
// device address comes from cudaGetSymbolAddress (device_setup below) and that is what the kernel is given.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
struct DeviceSetup {
  bool ready = false;
  unsigned char* scratch = nullptr;   // device address of g_static_scratch on this GPU
  int num_sms = 0;
};
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

int valid_uniform(double beta, double chi1, double chi2, double kq1, double kq2) {
  if (!(beta > 0.0) || !(beta <= 1.0)) return 0;
  if (!(chi1 >= 0.0) || !(chi1 <= 1.0) || !(chi2 >= 0.0) || !(chi2 <= 1.0)) return 0;
  return std::isfinite(kq1) && std::isfinite(kq2);
}

// The checks mc_create makes, without creating anything.
int valid_params(const mc_params* p) {
  if (!p || p->struct_size != sizeof(mc_params)) return 0;
  if (p->terms & ~63u) return 0;
  if (p->renorm_interval <= 0 || p->newton_iters < 1 || p->newton_iters > 16) return 0;
  if (p->integrator != MC_INTEG_RK4 && p->integrator != MC_INTEG_RK5) return 0;
  if (!(p->newton_tol >= 0.0) || !(p->r_merge >= 0.0) || !(p->r_escape > p->r_merge)) return 0;
  if (!(p->wait_budget_s > 0.0) || !(p->wait_budget_s <= 1e9)) return 0;
  if (p->per_orbit < 0 || p->per_orbit > 2) return 0;
  if (p->per_orbit == 1) return p->d_beta && p->d_chi1 && p->d_chi2 && p->d_kq1 && p->d_kq2;
  if (p->per_orbit == 2) return p->d_kq1 && p->d_kq2 && valid_uniform(p->beta, p->chi1, p->chi2, 1.0, 1.0);
  return valid_uniform(p->beta, p->chi1, p->chi2, p->kq1, p->kq2);
}

// Once per device, with that device current: resolve the scratch array's device address and read the SM count.
cudaError_t device_setup(int device, DeviceSetup* out) {
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  DeviceSetup& s = g_setup[device];
  if (!s.ready) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
    if (e != cudaSuccess) return e;
    if (major != 10) return cudaErrorNoKernelImageForDevice;   // the library holds sm_100a code only
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    unsigned char* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    s.scratch = ptr;
    s.num_sms = sms;
    s.ready = true;
  }
  *out = s;
  return cudaSuccess;
}

}  // namespace

extern "C" int mc_integrate_static(const mc_params* params, const double* states, int64_t n_orbits, double step_h,
                                   int64_t n_steps, int32_t correction_mode, double shadow_eps, double* out_states,
                                   double* out_invariants, double* out_fli, int32_t* out_status, int64_t* out_step) {
  // everything that can be refused is refused before the first CUDA call
  if (!valid_params(params)) return MC_EINVAL;
  if (params->terms & MC_TERM_RR) return MC_EINVAL;   // the dissipation integrals have no caller-side output here
  if (n_orbits < 0 || n_steps < 0 || n_steps > 0x7fffffffLL) return MC_EINVAL;
  if (correction_mode < 0 || correction_mode > 3) return MC_EINVAL;
  if (!std::isfinite(step_h) || !std::isfinite(shadow_eps)) return MC_EINVAL;
  const bool shadow = shadow_eps != 0.0;
  if (n_orbits > (int64_t)MC_STATIC_MAX_TRAJECTORIES) return MC_ELIMIT;
  const int64_t traj = n_orbits * (shadow ? 2 : 1);
  if (traj > (int64_t)MC_STATIC_MAX_TRAJECTORIES) return MC_ELIMIT;   // the fixed scratch has no room for more
  if (n_orbits > 0 && (!states || !out_states || !out_status || !out_step || (shadow && !out_fli))) return MC_EINVAL;
  if (params->device < 0 || params->device >= kMaxDevices) return MC_EINVAL;
  if (n_orbits == 0) return MC_OK;

  cudaError_t e = cudaSetDevice(params->device);
  DeviceSetup dev;
  if (e == cudaSuccess) e = device_setup(params->device, &dev);
  if (e == cudaErrorNoKernelImageForDevice) return MC_EARCH;
  if (e != cudaSuccess) return mc::record_cuda_failure(e);   // MC_ECUDA; mc_strerror(MC_ECUDA) then has the text
  cudaStream_t stream = (cudaStream_t)params->cuda_stream;

  McConsts uc;
  if (params->per_orbit == 1) memset(&uc, 0, sizeof(uc));
  else if (params->per_orbit == 2) mc_derive_consts(params->beta, params->chi1, params->chi2, 1.0, 1.0, params->terms, uc.v);
  else mc_derive_consts(params->beta, params->chi1, params->chi2, params->kq1, params->kq2, params->terms, uc.v);

  mc::IntegrateArgs A;
  memset(&A, 0, sizeof(A));
  A.beta = params->d_beta; A.chi1 = params->d_chi1; A.chi2 = params->d_chi2; A.kq1 = params->d_kq1; A.kq2 = params->d_kq2;
  A.terms = params->terms;
  A.renorm_interval = params->renorm_interval;
  A.newton_iters = params->newton_iters;
  A.newton_tol = params->newton_tol;
  A.integrator = params->integrator;
  A.r_merge2 = params->r_merge * params->r_merge;
  A.r_escape2 = params->r_escape * params->r_escape;
  A.wait_budget_ns = (unsigned long long)(params->wait_budget_s * 1e9);
  A.states = states; A.out_states = out_states; A.out_inv = out_invariants; A.out_fli = shadow ? out_fli : nullptr;
  A.out_status = out_status; A.out_step = out_step;
  A.n = n_orbits; A.n_steps = n_steps; A.h = step_h; A.hw = mc::step_weights(step_h); A.shadow_eps = shadow_eps;
  A.sample_interval = 1;
  // the scratch: queue header, then the per-orbit Gauss-Newton counters (written by the kernel, read by nobody here)
  A.queue = (unsigned long long*)dev.scratch;
  A.out_gn = (int64_t*)(dev.scratch + kQueueBytes);
  // one chunk: no `done` flags, no carry buffer
  A.n_units = (traj + 31) / 32;
  A.chunk_len = (int32_t)(n_steps > 0 ? n_steps : 1);
  A.n_chunks = 1;
  A.n_items = A.n_units;

  const bool qm = (params->terms & MC_TERM_QM) != 0;
  mc::LaunchFn fn = nullptr;
  switch (correction_mode) {
    case 0: fn = mc::launcher_mode0(params->per_orbit, qm, params->integrator, false); break;
    case 1: fn = mc::launcher_mode1(params->per_orbit, qm, params->integrator, false); break;
    case 2: fn = mc::launcher_mode2(params->per_orbit, qm, params->integrator, false); break;
    default: fn = mc::launcher_mode3(params->per_orbit, qm, params->integrator, false); break;
  }
  if (!fn) return MC_EINVAL;
  // The array keeps whatever the previous call left in it.  Only the queue header has to start at zero (the counters
  // are overwritten for every orbit of this batch); the memset is ordered on the caller's stream like the kernel.
  e = cudaMemsetAsync(dev.scratch, 0, kQueueBytes, stream);
  mc::KernelInfo ki;
  if (e == cudaSuccess) e = fn(uc, A, dev.num_sms, true, stream, &ki);
  if (e != cudaSuccess) return mc::record_cuda_failure(e);
  return MC_OK;
}
