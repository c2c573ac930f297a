// mc_flop_model.cpp -- mc_flop_model (include/mc_bench.h; built into benchlib/libmc_bench.so): the algorithmic operation counts of the kernels'
// own formulation, obtained by running the kernels' math templates (mc_math.cuh, mc_correct.cuh) once on the
// host with the counting scalar mc::Cnt.  Plain C++ (no CUDA): works on a box without a GPU.
#include <cstring>

#include "../include/mc_bench.h"
#include "mc_count.h"      // -I paper_1802_00147_b200/csrc: the kernels' own math templates
#include "mc_correct.cuh"

namespace {

struct HostConsts {
  double v[MC_NCONST];
  double operator[](int i) const { return v[i]; }
};

mc_op_counts delta(const mc::OpCounts& a, const mc::OpCounts& b) {
  mc_op_counts d;
  d.fma = a.fma - b.fma; d.mul = a.mul - b.mul; d.add = a.add - b.add; d.special = a.special - b.special;
  return d;
}
mc_op_counts sub(const mc_op_counts& a, const mc_op_counts& b) {
  mc_op_counts d = {a.fma - b.fma, a.mul - b.mul, a.add - b.add, a.special - b.special};
  return d;
}

// a generic bound orbit (config-0 like); the counts do not depend on the values
void sample_state(mc::Cnt* z) {
  const double v[12] = {20.0, 0.3, -0.2, 0.01, 0.2, 0.02, 0.6, 0.0, 0.8, 0.0, -0.6, -0.8};
  for (int i = 0; i < 12; ++i) z[i] = mc::Cnt(v[i]);
}

template <class F>
mc_op_counts count(F f) {
  const mc::OpCounts before = mc::op_counts();
  f();
  return delta(mc::op_counts(), before);
}

template <bool QM, int INTEG, bool RR>
void model(const HostConsts& c, int mode, int newton_iters, mc_flop_model_t* out) {
  using mc::Cnt;
  Cnt z[16], f[16];
  sample_state(z);
  out->rhs = count([&] { mc::pn_rhs<QM, RR>(c, z, f); });
  out->base_step = count([&] { mc::base_step<INTEG, QM, RR>(c, z, mc::step_weights(1.0), f); });
  mc::RefsT<Cnt> R;
  mc::references<QM>(c, z, R);
  out->references = count([&] { mc::references<QM>(c, z, R); });
  // correction: perturb the state a little so that the Gauss-Newton steps do not vanish
  auto run = [&](int iters) {
    Cnt y[12];
    for (int i = 0; i < 12; ++i) y[i] = Cnt(f[i].v * (1.0 + 1e-9 * (i + 1)));
    return count([&] {
      int gn = 0;
      if (mode == 1) mc::correct<1, QM>(c, y, R, iters, 0.0, gn);
      else if (mode == 2) mc::correct<2, QM>(c, y, R, iters, 1.0, gn);
      else if (mode == 3) mc::correct<3, QM>(c, y, R, iters, 0.0, gn);
    });
  };
  memset(&out->gn_step, 0, sizeof(out->gn_step));
  if (mode == 3) {
    const mc_op_counts c1 = run(1), c2 = run(2);
    out->gn_step = sub(c2, c1);
    out->correct_fixed = sub(c1, out->gn_step);
  } else {
    out->correct_fixed = run(newton_iters);
  }
  // status test of a completed step and one shadow renormalisation: the very templates the kernel's step loop calls
  // (mc_correct.cuh); the finite test is integer work, log10 is bookkeeping
  out->status = count([&] { (void)mc::radius_status(z, Cnt(4.0), Cnt(1e8)); });
  out->renorm = count([&] {
    Cnt y[12], acc = 0.0;
    for (int i = 0; i < 12; ++i) y[i] = Cnt(f[i].v);
    if (mode >= 1) mc::renormalise_shadow<1, QM>(c, y, z, Cnt(1e-8), acc, R);
    else mc::renormalise_shadow<0, QM>(c, y, z, Cnt(1e-8), acc, R);
  });
}

}  // namespace

extern "C" int mc_flop_model(uint32_t terms, int32_t correction_mode, int32_t integrator, int32_t newton_iters,
                             mc_flop_model_t* out) {
  if (!out || (terms & ~63u) || correction_mode < 0 || correction_mode > 3) return MC_EINVAL;
  if (integrator != MC_INTEG_RK4 && integrator != MC_INTEG_RK5) return MC_EINVAL;
  if (newton_iters < 1 || newton_iters > 16) return MC_EINVAL;
  HostConsts c;
  mc_derive_consts(0.8, 0.9, 0.7, 2.0, 3.0, terms, c.v);
  const bool qm = (terms & MC_TERM_QM) != 0;
  memset(out, 0, sizeof(*out));
  const bool rr = (terms & MC_TERM_RR) != 0, rk5 = integrator == MC_INTEG_RK5;
  if (rr) {
    if (qm) { if (rk5) model<true, 1, true>(c, correction_mode, newton_iters, out); else model<true, 0, true>(c, correction_mode, newton_iters, out); }
    else { if (rk5) model<false, 1, true>(c, correction_mode, newton_iters, out); else model<false, 0, true>(c, correction_mode, newton_iters, out); }
  } else {
    if (qm) { if (rk5) model<true, 1, false>(c, correction_mode, newton_iters, out); else model<true, 0, false>(c, correction_mode, newton_iters, out); }
    else { if (rk5) model<false, 1, false>(c, correction_mode, newton_iters, out); else model<false, 0, false>(c, correction_mode, newton_iters, out); }
  }
  return MC_OK;
}
