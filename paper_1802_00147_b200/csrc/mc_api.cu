// mc_api.cu -- the C ABI of include/mc.h: handle, validation, launches, host-buffer variant,
// evaluation entry point for the parity tests.  (The bench's instruments live in benchlib/, not here.)
#include <cuda_runtime.h>
#include <cub/device/device_radix_sort.cuh>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/mc.h"
#include "mc_kernel.cuh"
#include "mc_launch.h"

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error %d: %s", (int)e, cudaGetErrorString(e));
  return MC_ECUDA;
}
#define MC_CUDA(call)                               \
  do {                                              \
    cudaError_t e_ = (call);                        \
    if (e_ != cudaSuccess) return cuda_fail(e_);    \
  } while (0)

struct DeviceBuf {
  void* p = nullptr;
  size_t cap = 0;
  int reserve(size_t bytes) {
    if (bytes <= cap) return MC_OK;
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) return cuda_fail(e);
    cap = bytes;
    return MC_OK;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    cap = 0;
  }
};

}  // namespace

namespace mc {
int record_cuda_failure(cudaError_t e) { return cuda_fail(e); }
}  // namespace mc

struct mc_handle {
  mc_params P;
  McConsts uc;               // derived constants of the uniform parameter set
  cudaStream_t stream;
  int num_sms;
  int64_t last_n;            // orbits of the last mc_integrate (status buffers valid for these)
  DeviceBuf status, step, gn, diss;   // int32[n], int64[n], int64[n], double[4][n] (MC_TERM_RR)
  DeviceBuf sched, carry_d, carry_i, carry_g;   // work queue + per-unit flags; carried state between chunks
  DeviceBuf rg_keys, rg_idx, rg_tmp;            // mc_params.regroup: energy keys (2 x n doubles), slot -> orbit maps (2 x n int32), sort scratch
  DeviceBuf h_in, h_out, h_inv, h_fli;   // scratch of mc_integrate_host
  mc_launch_info info;
};

namespace {

int valid_scalars(double beta, double chi1, double chi2, double kq1, double kq2) {
  if (!(beta > 0.0) || !(beta <= 1.0)) return 0;            // m1 <= m2
  if (!(chi1 >= 0.0) || !(chi1 <= 1.0) || !(chi2 >= 0.0) || !(chi2 <= 1.0)) return 0;
  if (!std::isfinite(kq1) || !std::isfinite(kq2)) return 0;
  return 1;
}

// ---- evaluation kernel for mc_eval ---------------------------------------------------------------
template <int PARAMS, bool QM>
__global__ void __launch_bounds__(mc::kBlock)
eval_kernel(const __grid_constant__ McConsts uc, const __grid_constant__ mc::IntegrateArgs A, int what, int mode,
            const double* __restrict__ refs, double* __restrict__ out) {
  extern __shared__ double smem[];
  const int64_t t = (int64_t)blockIdx.x * mc::kBlock + threadIdx.x;
  const bool active = t < A.n;
  const int64_t o = active ? t : A.n - 1;
  using CP = typename mc::ConstsOf<PARAMS>::type;
  const CP c = mc::make_consts<PARAMS, CP>(uc, A, o, smem);
  double z[16], f[16];
#pragma unroll
  for (int i = 0; i < 12; ++i) z[i] = A.states[(int64_t)i * A.n + o];
  z[12] = z[13] = z[14] = z[15] = 0.0;
  int rows = 12;
  const bool rr = (A.terms & MC_TERM_RR) != 0;
  if (what == 0) {
    f[0] = mc::hamiltonian<QM>(c, z);
    rows = 1;
  } else if (what == 1) {
    if (rr) { mc::pn_rhs<QM, true>(c, z, f); rows = 16; }
    else mc::pn_rhs<QM, false>(c, z, f);
  } else if (what == 2) {
    mc::six_integrals<QM>(c, z, f);
    rows = 6;
  } else if (what == 3) {
    if (rr) {
      // fully per-orbit parameters + RK5 + 2.5PN is the one combination that is not built (register budget;
      // mc_integrate and mc_eval return MC_EINVAL for it)
      if constexpr (PARAMS != mc::PARAMS_PER_ORBIT) {
        if (A.integrator == 1) mc::rk5_step<QM, true>(c, z, A.hw, f);
        else mc::rk4_step<QM, true>(c, z, A.hw, f);
      } else {
        mc::rk4_step<QM, true>(c, z, A.hw, f);
      }
      rows = 16;
    } else if (A.integrator == 1) mc::rk5_step<QM, false>(c, z, A.hw, f);
    else mc::rk4_step<QM, false>(c, z, A.hw, f);
  } else {
    mc::Refs R;
    R.E0 = refs[o];
    R.J0[0] = refs[A.n + o]; R.J0[1] = refs[2 * A.n + o]; R.J0[2] = refs[3 * A.n + o];
    int gn;
    if (mode == 1) mc::correct<1, QM>(c, z, R, A.newton_iters, A.newton_tol, gn);
    else if (mode == 2) mc::correct<2, QM>(c, z, R, A.newton_iters, A.newton_tol, gn);
    else if (mode == 3) mc::correct<3, QM>(c, z, R, A.newton_iters, A.newton_tol, gn);
#pragma unroll
    for (int i = 0; i < 12; ++i) f[i] = z[i];
  }
  if (active) {
#pragma unroll
    for (int i = 0; i < 16; ++i)
      if (i < rows) out[(int64_t)i * A.n + o] = f[i];
  }
}

// ---- mc_params.regroup: energy of every orbit at t = 0 as a sort key ---------------------------------
// Orbits of equal energy have equal radial periods to 1PN order, so neighbours in energy order keep passing periastron
// together and a warp's lanes need their second Gauss-Newton step at the same steps.
template <int PARAMS, bool QM>
__global__ void __launch_bounds__(mc::kBlock)
energy_key_kernel(const __grid_constant__ McConsts uc, const __grid_constant__ mc::IntegrateArgs A, double* __restrict__ keys,
                  int32_t* __restrict__ idx) {
  extern __shared__ double smem[];
  const int64_t t = (int64_t)blockIdx.x * mc::kBlock + threadIdx.x;
  const bool active = t < A.n;
  const int64_t o = active ? t : A.n - 1;
  using CP = typename mc::ConstsOf<PARAMS>::type;
  const CP c = mc::make_consts<PARAMS, CP>(uc, A, o, smem);
  double z[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) z[i] = A.states[(int64_t)i * A.n + o];
  const double H = mc::hamiltonian<QM>(c, z);
  if (active) {
    keys[t] = H;
    idx[t] = (int32_t)t;
  }
}

void fill_args(const mc_handle* h, mc::IntegrateArgs& A) {
  memset(&A, 0, sizeof(A));
  A.beta = h->P.d_beta; A.chi1 = h->P.d_chi1; A.chi2 = h->P.d_chi2; A.kq1 = h->P.d_kq1; A.kq2 = h->P.d_kq2;
  A.terms = h->P.terms;
  A.renorm_interval = h->P.renorm_interval;
  A.newton_iters = h->P.newton_iters;
  A.newton_tol = h->P.newton_tol;
  A.integrator = h->P.integrator;
  A.r_merge2 = h->P.r_merge * h->P.r_merge;
  A.r_escape2 = h->P.r_escape * h->P.r_escape;
  A.wait_budget_ns = (unsigned long long)(h->P.wait_budget_s * 1e9);
}

}  // namespace

extern "C" {

int mc_params_default(mc_params* p) {
  if (!p) return MC_EINVAL;
  memset(p, 0, sizeof(*p));
  p->struct_size = (uint32_t)sizeof(mc_params);
  p->terms = MC_TERM_1PN | MC_TERM_2PN | MC_TERM_SO | MC_TERM_S1S2;
  p->device = 0;
  p->per_orbit = 0;
  p->beta = p->chi1 = p->chi2 = p->kq1 = p->kq2 = 1.0;
  p->renorm_interval = 100;
  p->newton_iters = 4;
  p->newton_tol = 1e-10;
  p->r_merge = 2.0;
  p->r_escape = 1e4;
  p->cuda_stream = nullptr;
  p->chunk_steps = 0;
  p->integrator = MC_INTEG_RK4;
  p->wait_budget_s = 600.0;
  p->regroup = 0;
  return MC_OK;
}

int mc_create(const mc_params* params, mc_handle** out_handle) {
  if (!params || !out_handle) return MC_EINVAL;
  if (params->struct_size != sizeof(mc_params)) return MC_EINVAL;
  if (params->terms & ~63u) return MC_EINVAL;
  if (params->renorm_interval <= 0 || params->newton_iters < 1 || params->newton_iters > 16) return MC_EINVAL;
  if (params->chunk_steps < 0) return MC_EINVAL;
  if (params->integrator != MC_INTEG_RK4 && params->integrator != MC_INTEG_RK5) return MC_EINVAL;
  if (!(params->newton_tol >= 0.0) || !(params->r_merge >= 0.0) || !(params->r_escape > params->r_merge)) return MC_EINVAL;
  if (!(params->wait_budget_s > 0.0) || !(params->wait_budget_s <= 1e9)) return MC_EINVAL;
  if (params->regroup != 0 && params->regroup != 1) return MC_EINVAL;
  if (params->per_orbit < 0 || params->per_orbit > 2) return MC_EINVAL;
  if (params->per_orbit == 1) {
    if (!params->d_beta || !params->d_chi1 || !params->d_chi2 || !params->d_kq1 || !params->d_kq2) return MC_EINVAL;
  } else if (params->per_orbit == 2) {
    if (!params->d_kq1 || !params->d_kq2 || !valid_scalars(params->beta, params->chi1, params->chi2, 1.0, 1.0)) return MC_EINVAL;
  } else if (!valid_scalars(params->beta, params->chi1, params->chi2, params->kq1, params->kq2)) {
    return MC_EINVAL;
  }
  int ndev = 0;
  MC_CUDA(cudaGetDeviceCount(&ndev));
  if (params->device < 0 || params->device >= ndev) return MC_EINVAL;
  cudaDeviceProp prop;
  MC_CUDA(cudaGetDeviceProperties(&prop, params->device));
  if (prop.major != 10) return MC_EARCH;   // the fat binary holds sm_100a SASS only
  MC_CUDA(cudaSetDevice(params->device));
  mc_handle* h = new (std::nothrow) mc_handle();
  if (!h) return MC_ENOMEM;
  h->P = *params;
  h->stream = (cudaStream_t)params->cuda_stream;
  h->num_sms = prop.multiProcessorCount;
  h->last_n = 0;
  memset(&h->info, 0, sizeof(h->info));
  if (params->per_orbit == 1) memset(&h->uc, 0, sizeof(h->uc));
  else if (params->per_orbit == 2)   // the kappa-dependent constants (q_i, m_ii) are linear in kappa: derived with kappa = 1
    mc_derive_consts(params->beta, params->chi1, params->chi2, 1.0, 1.0, params->terms, h->uc.v);
  else mc_derive_consts(params->beta, params->chi1, params->chi2, params->kq1, params->kq2, params->terms, h->uc.v);
  *out_handle = h;
  return MC_OK;
}

static int integrate_impl(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                          int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                          double* out_fli, int64_t sample_interval, double* out_samples, void* user_carry, int32_t resume);

int mc_integrate(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                 int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                 double* out_fli) {
  return integrate_impl(h, states, n_orbits, step_h, n_steps, correction_mode, shadow_eps, out_states,
                        out_invariants, out_fli, 0, nullptr, nullptr, 0);
}

int mc_integrate_sampled(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                         int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                         double* out_fli, int64_t sample_interval, double* out_samples) {
  return integrate_impl(h, states, n_orbits, step_h, n_steps, correction_mode, shadow_eps, out_states,
                        out_invariants, out_fli, sample_interval, out_samples, nullptr, 0);
}

int64_t mc_carry_bytes(int64_t n_orbits, int32_t with_shadow) {
  if (n_orbits < 0) return MC_EINVAL;
  const int64_t tp = ((n_orbits * (with_shadow ? 2 : 1) + 31) / 32) * 32;
  return tp * (int64_t)(17 * sizeof(double) + 2 * sizeof(unsigned long long) + 2 * sizeof(int32_t));
}

int mc_integrate_ex(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                    int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                    double* out_fli, void* carry, int32_t resume) {
  if (!carry && n_orbits > 0) return MC_EINVAL;
  if (resume != 0 && resume != 1) return MC_EINVAL;
  return integrate_impl(h, states, n_orbits, step_h, n_steps, correction_mode, shadow_eps, out_states,
                        out_invariants, out_fli, 0, nullptr, carry, resume);
}

static int integrate_impl(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                          int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                          double* out_fli, int64_t sample_interval, double* out_samples, void* user_carry, int32_t resume) {
  if (sample_interval < 0 || sample_interval > 0x7fffffffLL || (sample_interval > 0 && !out_samples && n_orbits > 0)) return MC_EINVAL;
  if (!h || n_orbits < 0 || n_steps < 0 || n_steps > 0x7fffffffLL) return MC_EINVAL;
  if (correction_mode < 0 || correction_mode > 3) return MC_EINVAL;
  if (!std::isfinite(step_h) || !std::isfinite(shadow_eps)) return MC_EINVAL;
  const bool shadow = shadow_eps != 0.0;
  if (n_orbits > 0 && ((!states && !resume) || !out_states || (shadow && !out_fli))) return MC_EINVAL;
  if (n_orbits > (int64_t)1 << 40) return MC_EINVAL;
  // everything that can be refused is refused before the handle's record of the last launch (last_n) is touched:
  // after a failed call mc_get_status / mc_get_work still describe the last launch that did run
  const bool qm = (h->P.terms & MC_TERM_QM) != 0;
  const bool rr = (h->P.terms & MC_TERM_RR) != 0;
  mc::LaunchFn fn = nullptr;
  switch (correction_mode) {
    case 0: fn = mc::launcher_mode0(h->P.per_orbit, qm, h->P.integrator, rr); break;
    case 1: fn = mc::launcher_mode1(h->P.per_orbit, qm, h->P.integrator, rr); break;
    case 2: fn = mc::launcher_mode2(h->P.per_orbit, qm, h->P.integrator, rr); break;
    default: fn = mc::launcher_mode3(h->P.per_orbit, qm, h->P.integrator, rr); break;
  }
  if (!fn) return MC_EINVAL;   // per_orbit = 1 with RK5 and MC_TERM_RR: not built (register budget; include/mc.h)
  const int64_t traj = n_orbits * (shadow ? 2 : 1);
  if ((traj + 31) / 32 > 0x3fffffffLL) return MC_EINVAL;
  MC_CUDA(cudaSetDevice(h->P.device));
  if (n_orbits == 0) { h->last_n = 0; return MC_OK; }
  h->last_n = 0;               // until the launch below has been enqueued the status buffers describe nothing
  int rc = h->status.reserve(sizeof(int32_t) * (size_t)n_orbits);
  if (rc) return rc;
  rc = h->step.reserve(sizeof(int64_t) * (size_t)n_orbits);
  if (rc) return rc;
  rc = h->gn.reserve(sizeof(int64_t) * (size_t)n_orbits);
  if (rc) return rc;
  if (rr && (rc = h->diss.reserve(sizeof(double) * 4 * (size_t)n_orbits))) return rc;

  mc::IntegrateArgs A;
  fill_args(h, A);
  A.states = states; A.out_states = out_states; A.out_inv = out_invariants; A.out_fli = shadow ? out_fli : nullptr;
  A.out_status = (int32_t*)h->status.p; A.out_step = (int64_t*)h->step.p; A.out_gn = (int64_t*)h->gn.p;
  A.out_diss = rr ? (double*)h->diss.p : nullptr;
  A.n = n_orbits; A.n_steps = n_steps; A.h = step_h; A.hw = mc::step_weights(step_h); A.shadow_eps = shadow_eps;
  A.samples = sample_interval > 0 ? out_samples : nullptr;
  A.sample_interval = sample_interval > 0 ? (int32_t)sample_interval : 1;

  A.n_units = (traj + 31) / 32;
  A.chunk_len = 1; A.n_chunks = 1; A.n_items = A.n_units;
  mc::KernelInfo ki;
  MC_CUDA(fn(h->uc, A, h->num_sms, false, h->stream, &ki));                  // occupancy / register query
  // Chunking policy: one chunk when every unit is resident at once (nothing to balance)
  // or the run is short; otherwise about 128 chunks of >= 256 steps, a multiple of renorm_interval.
  const int64_t slots = (int64_t)h->num_sms * ki.blocks_per_sm * (mc::kBlock / 32);
  int64_t chunk = n_steps > 0 ? n_steps : 1;
  if (h->P.chunk_steps > 0) {
    chunk = h->P.chunk_steps;
  } else if (A.n_units > slots && n_steps >= 512) {
    chunk = (n_steps + 127) / 128;
    if (chunk < 256) chunk = 256;
    const int64_t ri = h->P.renorm_interval;
    if (shadow) chunk = ((chunk + ri - 1) / ri) * ri;
  }
  if (chunk > 0x7fffffffLL) chunk = 0x7fffffffLL;
  // the kernel counts the Gauss-Newton steps and warp passes of ONE work item in 32 bits (at most newton_iters per
  // step) and adds them to 64-bit totals at chunk boundaries: keep chunk_len * newton_iters below 2^32
  const int64_t counter_cap = 0xffffffffLL / h->P.newton_iters;
  if (chunk > counter_cap) chunk = counter_cap;
  int64_t n_chunks = n_steps > 0 ? (n_steps + chunk - 1) / chunk : 1;
  if (n_chunks > 0x7fffffffLL) return MC_EINVAL;
  A.chunk_len = (int32_t)chunk;
  A.n_chunks = (int32_t)n_chunks;
  A.n_items = A.n_units * n_chunks;
  rc = h->sched.reserve(32 + sizeof(int32_t) * (size_t)A.n_units);
  if (rc) return rc;
  A.queue = (unsigned long long*)h->sched.p;
  A.done = (int32_t*)((char*)h->sched.p + 32);
  A.resume = resume; A.save_final = user_carry ? 1 : 0;
  if (user_carry) {
    // caller-owned checkpoint (mc_carry_bytes): [17][tp] doubles, [2][tp] u64, [2][tp] int32 -- also the chunk carry
    const size_t tp = (size_t)A.n_units * 32;
    A.carry_d = (double*)user_carry;
    A.carry_g = (unsigned long long*)(A.carry_d + 17 * tp);
    A.carry_i = (int32_t*)(A.carry_g + 2 * tp);
  } else if (n_chunks > 1) {
    const size_t tp = (size_t)A.n_units * 32;
    if ((rc = h->carry_d.reserve(sizeof(double) * 17 * tp))) return rc;
    if ((rc = h->carry_i.reserve(sizeof(int32_t) * 2 * tp))) return rc;
    if ((rc = h->carry_g.reserve(sizeof(unsigned long long) * 2 * tp))) return rc;
    A.carry_d = (double*)h->carry_d.p; A.carry_i = (int32_t*)h->carry_i.p; A.carry_g = (unsigned long long*)h->carry_g.p;
  }
  A.perm = nullptr;
  if (h->P.regroup && !user_carry && sample_interval == 0 && n_orbits >= 64 && n_orbits <= 0x7fffffffLL) {
    // slot -> orbit map: orbits in order of their energy at t = 0 (stable radix sort; device-side, stream-ordered)
    const size_t n = (size_t)n_orbits;
    if ((rc = h->rg_keys.reserve(sizeof(double) * 2 * n))) return rc;
    if ((rc = h->rg_idx.reserve(sizeof(int32_t) * 2 * n))) return rc;
    double* k_in = (double*)h->rg_keys.p;
    double* k_out = k_in + n;
    int32_t* i_in = (int32_t*)h->rg_idx.p;
    int32_t* i_out = i_in + n;
    size_t tmp_bytes = 0;
    MC_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, k_in, k_out, i_in, i_out, (int)n_orbits, 0, 64, h->stream));
    if ((rc = h->rg_tmp.reserve(tmp_bytes))) return rc;
    const int kgrid = (int)((n_orbits + mc::kBlock - 1) / mc::kBlock);
    const int kp = h->P.per_orbit == 1 ? 1 : ((h->P.per_orbit == 2 && qm) ? 2 : 0);
    const size_t ksmem = kp == 1 ? sizeof(double) * MC_NCONST * mc::kBlock : 0;
    if (ksmem > 48 * 1024) {
      MC_CUDA(cudaFuncSetAttribute(energy_key_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ksmem));
      MC_CUDA(cudaFuncSetAttribute(energy_key_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ksmem));
    }
    if (kp == 1 && qm) energy_key_kernel<1, true><<<kgrid, mc::kBlock, ksmem, h->stream>>>(h->uc, A, k_in, i_in);
    else if (kp == 1) energy_key_kernel<1, false><<<kgrid, mc::kBlock, ksmem, h->stream>>>(h->uc, A, k_in, i_in);
    else if (kp == 2) energy_key_kernel<2, true><<<kgrid, mc::kBlock, 0, h->stream>>>(h->uc, A, k_in, i_in);
    else if (qm) energy_key_kernel<0, true><<<kgrid, mc::kBlock, 0, h->stream>>>(h->uc, A, k_in, i_in);
    else energy_key_kernel<0, false><<<kgrid, mc::kBlock, 0, h->stream>>>(h->uc, A, k_in, i_in);
    MC_CUDA(cudaGetLastError());
    MC_CUDA(cub::DeviceRadixSort::SortPairs(h->rg_tmp.p, tmp_bytes, k_in, k_out, i_in, i_out, (int)n_orbits, 0, 64, h->stream));
    A.perm = i_out;
  }
  MC_CUDA(cudaMemsetAsync(h->sched.p, 0, 32 + sizeof(int32_t) * (size_t)A.n_units, h->stream));
  MC_CUDA(fn(h->uc, A, h->num_sms, true, h->stream, &ki));
  h->info.grid = ki.grid;
  h->info.chunk_steps = A.chunk_len;
  h->info.n_chunks = A.n_chunks;
  h->info.block = ki.block;
  h->info.regs_per_thread = ki.regs;
  h->info.local_bytes = ki.local_bytes;
  h->info.blocks_per_sm = ki.blocks_per_sm;
  h->info.num_sms = h->num_sms;
  h->info.smem_bytes = (int32_t)ki.smem;
  const int kparams = (h->P.per_orbit == 2 && !qm) ? 0 : h->P.per_orbit;   // kappa is unused without the QM term
  h->info.variant = (kparams == 1 ? 1 : 0) | (qm ? 2 : 0) | (kparams == 2 ? 4 : 0) | (rr ? 8 : 0) | (correction_mode << 4) | (h->P.integrator << 8) | (A.perm ? 1024 : 0);
  h->info.trajectories = traj;
  h->last_n = n_orbits;
  return MC_OK;
}

int mc_get_status(mc_handle* h, int32_t* out_status, int64_t* out_step) {
  if (!h) return MC_EINVAL;
  if (h->last_n == 0) return MC_OK;
  MC_CUDA(cudaSetDevice(h->P.device));
  if (out_status)
    MC_CUDA(cudaMemcpyAsync(out_status, h->status.p, sizeof(int32_t) * (size_t)h->last_n, cudaMemcpyDeviceToDevice, h->stream));
  if (out_step)
    MC_CUDA(cudaMemcpyAsync(out_step, h->step.p, sizeof(int64_t) * (size_t)h->last_n, cudaMemcpyDeviceToDevice, h->stream));
  return MC_OK;
}

int mc_get_work(mc_handle* h, int64_t* out_gn_steps) {
  if (!h || !out_gn_steps) return MC_EINVAL;
  if (h->last_n == 0) return MC_OK;
  MC_CUDA(cudaSetDevice(h->P.device));
  MC_CUDA(cudaMemcpyAsync(out_gn_steps, h->gn.p, sizeof(int64_t) * (size_t)h->last_n, cudaMemcpyDeviceToDevice, h->stream));
  return MC_OK;
}

int mc_get_warp_work(mc_handle* h, int64_t* out_host2) {
  if (!h || !out_host2) return MC_EINVAL;
  out_host2[0] = out_host2[1] = 0;
  if (h->last_n == 0 || !h->sched.p) return MC_OK;
  MC_CUDA(cudaSetDevice(h->P.device));
  MC_CUDA(cudaMemcpyAsync(out_host2, (char*)h->sched.p + 8, 2 * sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
  MC_CUDA(cudaStreamSynchronize(h->stream));
  return MC_OK;
}

int mc_debug_check(mc_handle* h, int64_t* out_line) {
  if (!h || !out_line) return MC_EINVAL;
#ifndef MC_CHECKED
  *out_line = -1;
  return MC_OK;
#else
  *out_line = 0;
  if (h->last_n == 0 || !h->sched.p) return MC_OK;
  MC_CUDA(cudaSetDevice(h->P.device));
  MC_CUDA(cudaMemcpyAsync(out_line, (char*)h->sched.p + 24, sizeof(int64_t), cudaMemcpyDeviceToHost, h->stream));
  MC_CUDA(cudaStreamSynchronize(h->stream));
  return MC_OK;
#endif
}

int mc_get_dissipation(mc_handle* h, double* out_wg) {
  if (!h || !out_wg) return MC_EINVAL;
  if (!(h->P.terms & MC_TERM_RR)) return MC_EINVAL;
  if (h->last_n == 0) return MC_OK;
  MC_CUDA(cudaSetDevice(h->P.device));
  MC_CUDA(cudaMemcpyAsync(out_wg, h->diss.p, sizeof(double) * 4 * (size_t)h->last_n, cudaMemcpyDeviceToDevice, h->stream));
  return MC_OK;
}

int mc_integrate_host(mc_handle* h, const double* states, int64_t n_orbits, double step_h, int64_t n_steps,
                      int32_t correction_mode, double shadow_eps, double* out_states, double* out_invariants,
                      double* out_fli, int32_t* out_status, int64_t* out_step) {
  if (!h || n_orbits < 0) return MC_EINVAL;
  const bool shadow = shadow_eps != 0.0;
  if (n_orbits > 0 && (!states || !out_states || (shadow && !out_fli))) return MC_EINVAL;
  if (n_orbits == 0) { h->last_n = 0; return MC_OK; }
  MC_CUDA(cudaSetDevice(h->P.device));
  const size_t sb = sizeof(double) * 12 * (size_t)n_orbits;
  int rc;
  if ((rc = h->h_in.reserve(sb))) return rc;
  if ((rc = h->h_out.reserve(sb))) return rc;
  if (out_invariants && (rc = h->h_inv.reserve(sb))) return rc;
  if (shadow && (rc = h->h_fli.reserve(sizeof(double) * (size_t)n_orbits))) return rc;
  MC_CUDA(cudaMemcpyAsync(h->h_in.p, states, sb, cudaMemcpyHostToDevice, h->stream));
  rc = mc_integrate(h, (const double*)h->h_in.p, n_orbits, step_h, n_steps, correction_mode, shadow_eps,
                    (double*)h->h_out.p, out_invariants ? (double*)h->h_inv.p : nullptr,
                    shadow ? (double*)h->h_fli.p : nullptr);
  if (rc) return rc;
  MC_CUDA(cudaMemcpyAsync(out_states, h->h_out.p, sb, cudaMemcpyDeviceToHost, h->stream));
  if (out_invariants) MC_CUDA(cudaMemcpyAsync(out_invariants, h->h_inv.p, sb, cudaMemcpyDeviceToHost, h->stream));
  if (shadow) MC_CUDA(cudaMemcpyAsync(out_fli, h->h_fli.p, sizeof(double) * (size_t)n_orbits, cudaMemcpyDeviceToHost, h->stream));
  if (out_status) MC_CUDA(cudaMemcpyAsync(out_status, h->status.p, sizeof(int32_t) * (size_t)n_orbits, cudaMemcpyDeviceToHost, h->stream));
  if (out_step) MC_CUDA(cudaMemcpyAsync(out_step, h->step.p, sizeof(int64_t) * (size_t)n_orbits, cudaMemcpyDeviceToHost, h->stream));
  MC_CUDA(cudaStreamSynchronize(h->stream));
  return MC_OK;
}

int mc_eval(mc_handle* h, int32_t what, const double* states, int64_t n, double step_h, int32_t mode,
            const double* refs, double* out) {
  if (!h || n < 0 || what < 0 || what > 4) return MC_EINVAL;
  if (n == 0) return MC_OK;
  if (!states || !out) return MC_EINVAL;
  if (what == 4 && (mode < 0 || mode > 3 || !refs)) return MC_EINVAL;   // the kernel reads refs for every mode
  if (what == 3 && h->P.per_orbit == 1 && h->P.integrator == 1 && (h->P.terms & MC_TERM_RR)) return MC_EINVAL;   // not built
  MC_CUDA(cudaSetDevice(h->P.device));
  mc::IntegrateArgs A;
  fill_args(h, A);
  A.states = states; A.n = n; A.h = step_h; A.hw = mc::step_weights(step_h);
  const bool qm = (h->P.terms & MC_TERM_QM) != 0, po = h->P.per_orbit == 1, ka = h->P.per_orbit == 2 && qm;
  const int grid = (int)((n + mc::kBlock - 1) / mc::kBlock);
  const size_t smem = po ? sizeof(double) * MC_NCONST * mc::kBlock : 0;
  if (po && qm) eval_kernel<1, true><<<grid, mc::kBlock, smem, h->stream>>>(h->uc, A, what, mode, refs, out);
  else if (po) eval_kernel<1, false><<<grid, mc::kBlock, smem, h->stream>>>(h->uc, A, what, mode, refs, out);
  else if (ka) eval_kernel<2, true><<<grid, mc::kBlock, smem, h->stream>>>(h->uc, A, what, mode, refs, out);
  else if (qm) eval_kernel<0, true><<<grid, mc::kBlock, smem, h->stream>>>(h->uc, A, what, mode, refs, out);
  else eval_kernel<0, false><<<grid, mc::kBlock, smem, h->stream>>>(h->uc, A, what, mode, refs, out);
  MC_CUDA(cudaGetLastError());
  return MC_OK;
}

int mc_last_launch_info(mc_handle* h, mc_launch_info* out) {
  if (!h || !out) return MC_EINVAL;
  *out = h->info;
  return MC_OK;
}

int mc_destroy(mc_handle* h) {
  if (!h) return MC_EINVAL;
  cudaSetDevice(h->P.device);
  h->status.release(); h->step.release(); h->gn.release(); h->diss.release();
  h->sched.release(); h->carry_d.release(); h->carry_i.release(); h->carry_g.release();
  h->rg_keys.release(); h->rg_idx.release(); h->rg_tmp.release();
  h->h_in.release(); h->h_out.release(); h->h_inv.release(); h->h_fli.release();
  delete h;
  return MC_OK;
}

const char* mc_strerror(int code) {
  switch (code) {
    case MC_OK: return "ok";
    case MC_EINVAL: return "invalid argument";
    case MC_ECUDA: return g_cuda_msg;
    case MC_EARCH: return "device is not compute capability 10.x (library holds sm_100a code only)";
    case MC_ENOMEM: return "host allocation failed";
    case MC_ELIMIT: return "batch too large for mc_integrate_static: its fixed device scratch holds at most 32768 trajectories (orbits, or 2 x orbits with a shadow); use mc_integrate";
    default: return "unknown mc_error";
  }
}

}  // extern "C"
