// pn_oracle_capi.cpp -- C entry points of the CPU ORACLE (test infrastructure,
// NOT the product; see pn_oracle.hpp).  Arrays are plain double, SoA [12][n]
// (rx ry rz px py pz s1x s1y s1z s2x s2y s2z), the same layout as include/mc.h,
// so a test hands the same numpy arrays to both sides.
//
// precision: 0 = long double (parity oracle), 1 = double (timed CPU baseline).
// Build: oracle/build.py (g++ -O2 -fopenmp, no fast-math).
#include "pn_oracle.hpp"

#include <omp.h>

#include <cstring>

namespace pn_oracle {

// Flop-counting scalar: every +,-,*,/ and sqrt counts 1 (log10, comparisons: 0).
struct Counted {
  double v;
  static thread_local long long flops;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  Counted(int x) : v(x) {}
};
thread_local long long Counted::flops = 0;
inline Counted operator+(Counted a, Counted b) { ++Counted::flops; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { ++Counted::flops; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { ++Counted::flops; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { ++Counted::flops; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline bool operator<(Counted a, Counted b) { return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { return a.v >= b.v; }
inline bool operator==(Counted a, Counted b) { return a.v == b.v; }
inline Counted o_sqrt(Counted x) { ++Counted::flops; return Counted(sqrt(x.v)); }
inline Counted o_log10(Counted x) { return Counted(log10(x.v)); }
inline Counted o_abs(Counted x) { return Counted(fabs(x.v)); }
inline bool o_finite(Counted x) { return std::isfinite(x.v); }
inline double to_double(Counted x) { return x.v; }
inline double to_double(long double x) { return (double)x; }
inline double to_double(double x) { return x; }

template <class T> State<T> load_state(const double* s, int64_t n, int64_t i) {
  auto g = [&](int c) { return T(s[(int64_t)c * n + i]); };
  return {{g(0), g(1), g(2)}, {g(3), g(4), g(5)}, {g(6), g(7), g(8)}, {g(9), g(10), g(11)}, {T(0.0), {T(0.0), T(0.0), T(0.0)}}};
}
// rows 12-15 of a [16][n] array: W, Gx, Gy, Gz (the dissipation integrals / their time derivatives)
template <class T> void store_diss(double* s, int64_t n, int64_t i, const Diss<T>& d) {
  const T v[4] = {d.w, d.g.x, d.g.y, d.g.z};
  for (int c = 0; c < 4; ++c) s[(int64_t)(12 + c) * n + i] = to_double(v[c]);
}
template <class T> void store_state(double* s, int64_t n, int64_t i, const State<T>& z) {
  const T v[12] = {z.r.x, z.r.y, z.r.z, z.p.x, z.p.y, z.p.z, z.s1.x, z.s1.y, z.s1.z, z.s2.x, z.s2.y, z.s2.z};
  for (int c = 0; c < 12; ++c) s[(int64_t)c * n + i] = to_double(v[c]);
}
template <class T>
Params<T> load_params(const double* beta, const double* chi1, const double* chi2, const double* kq1,
                      const double* kq2, uint32_t terms, int64_t i) {
  return {T(beta[i]), T(chi1[i]), T(chi2[i]), T(kq1[i]), T(kq2[i]), terms};
}

struct ParamArrays { const double *beta, *chi1, *chi2, *kq1, *kq2; uint32_t terms; };

// what: 0 H -> out[1][n]; 1 J -> out[3][n]; 2 rhs -> out[12][n];
// 3 gradient (dH/dr, dH/dp, dH/dS1, dH/dS2) -> out[12][n]; 4 six integrals -> out[6][n]; 5 rhs + (dW/dt, dG/dt) -> out[16][n]
template <class T> void eval_t(int what, int64_t n, const double* states, const ParamArrays& A, double* out) {
  for (int64_t i = 0; i < n; ++i) {
    const State<T> z = load_state<T>(states, n, i);
    const Params<T> P = load_params<T>(A.beta, A.chi1, A.chi2, A.kq1, A.kq2, A.terms, i);
    if (what == 0) {
      out[i] = to_double(hamiltonian(z, P));
    } else if (what == 1) {
      const V3<T> J = total_J(z, P);
      out[i] = to_double(J.x); out[n + i] = to_double(J.y); out[2 * n + i] = to_double(J.z);
    } else if (what == 2) {
      store_state(out, n, i, rhs(z, P));
    } else if (what == 3) {
      const Grad<T> g = gradient(z, P);
      store_state(out, n, i, State<T>{g.dHdr, g.dHdp, g.dHdS1, g.dHdS2, z.d});
    } else if (what == 5) {   // rhs with the dissipation rates: out[16][n], rows 12-15 = dW/dt, dG/dt
      const State<T> f = rhs(z, P);
      store_state(out, n, i, f);
      store_diss(out, n, i, f.d);
    } else {
      T v[6];
      six_integrals(z, P, v);
      for (int c = 0; c < 6; ++c) out[(int64_t)c * n + i] = to_double(v[c]);
    }
  }
}

template <class T>
void step_t(int64_t n, const double* states, const ParamArrays& A, double h, int integrator, double* out) {
  for (int64_t i = 0; i < n; ++i)
    store_state(out, n, i, base_step(load_state<T>(states, n, i),
                                     T(h), load_params<T>(A.beta, A.chi1, A.chi2, A.kq1, A.kq2, A.terms, i), integrator));
}

template <class T>
void correct_t(int64_t n, const double* states, const ParamArrays& A, const double* E0, const double* J0,
               int mode, int newton_iters, double newton_tol, double* out, int32_t* ok) {
  for (int64_t i = 0; i < n; ++i) {
    State<T> z = load_state<T>(states, n, i);
    const Params<T> P = load_params<T>(A.beta, A.chi1, A.chi2, A.kq1, A.kq2, A.terms, i);
    const Refs<T> R = {T(E0[i]), {T(J0[i]), T(J0[n + i]), T(J0[2 * n + i])}};
    const bool r = correct(z, P, R, mode, newton_iters, T(newton_tol));
    if (ok) ok[i] = r ? 1 : 0;
    store_state(out, n, i, z);
  }
}

template <class T>
void integrate_t(int64_t n, const double* states, const ParamArrays& A, double h, int64_t n_steps,
                 double shadow_eps, const Options& O, double* out_states, double* out_inv, double* out_fli,
                 int32_t* out_status, int64_t* out_step, int64_t* out_gn, int n_threads,
                 int64_t sample_interval, double* out_samples, double* out_shadow, double* out_diss) {
#pragma omp parallel for schedule(static) num_threads(n_threads)
  for (int64_t i = 0; i < n; ++i) {
    const State<T> z = load_state<T>(states, n, i);
    const Params<T> P = load_params<T>(A.beta, A.chi1, A.chi2, A.kq1, A.kq2, A.terms, i);
    // samples: [n_steps / sample_interval][12][n], the layout of include/mc.h
    auto sampler = [&](int64_t s, const State<T>& zz) { store_state(out_samples + s * 12 * n, n, i, zz); };
    const OrbitResult<T> R = integrate_orbit<T>(z, P, T(h), n_steps, T(shadow_eps), O,
                                                out_samples ? sample_interval : 0, sampler);
    if (out_states) store_state(out_states, n, i, R.z);
    if (out_inv)
      for (int c = 0; c < 6; ++c) {
        out_inv[(int64_t)c * n + i] = to_double(R.inv0[c]);
        out_inv[(int64_t)(6 + c) * n + i] = to_double(R.inv1[c]);
      }
    if (out_fli) out_fli[i] = to_double(R.fli);
    if (out_status) out_status[i] = R.status;
    if (out_step) out_step[i] = R.steps_done;
    if (out_gn) out_gn[i] = R.gn_steps;
    if (out_diss) {     // [4][n]: W, Gx, Gy, Gz of the orbit at the end of the run
      const T v[4] = {R.z.d.w, R.z.d.g.x, R.z.d.g.y, R.z.d.g.z};
      for (int c = 0; c < 4; ++c) out_diss[(int64_t)c * n + i] = to_double(v[c]);
    }
    if (out_shadow) {   // [16][n]: the shadow's final state, then E0', J0' (the integrals it is corrected onto)
      store_state(out_shadow, n, i, R.zs);
      const T refs[4] = {R.Es0, R.Js0.x, R.Js0.y, R.Js0.z};
      for (int c = 0; c < 4; ++c) out_shadow[(int64_t)(12 + c) * n + i] = to_double(refs[c]);
    }
  }
}

}  // namespace pn_oracle

using namespace pn_oracle;

extern "C" {

int oracle_eval(int precision, int what, int64_t n, const double* states, const double* beta,
                const double* chi1, const double* chi2, const double* kq1, const double* kq2,
                uint32_t terms, double* out) {
  const ParamArrays A = {beta, chi1, chi2, kq1, kq2, terms};
  if (precision == 0) eval_t<long double>(what, n, states, A, out);
  else eval_t<double>(what, n, states, A, out);
  return 0;
}

int oracle_rk4_step(int precision, int64_t n, const double* states, const double* beta, const double* chi1,
                    const double* chi2, const double* kq1, const double* kq2, uint32_t terms, double h,
                    int integrator, double* out) {
  const ParamArrays A = {beta, chi1, chi2, kq1, kq2, terms};
  if (precision == 0) step_t<long double>(n, states, A, h, integrator, out);
  else step_t<double>(n, states, A, h, integrator, out);
  return 0;
}

// The Butcher tableau the oracle integrates with (integrator 0 / 1): c[s], a[s*s] row-major, b[s]; returns s.
int oracle_tableau(int integrator, double* c, double* a, double* b) {
  const Tableau& T = integrator == 1 ? tableau_rk5() : tableau_rk4();
  for (int i = 0; i < T.stages; ++i) { c[i] = T.c[i]; b[i] = T.b[i]; }
  for (int i = 0; i < T.stages * T.stages; ++i) a[i] = T.a[i];
  return T.stages;
}

int oracle_correct(int precision, int64_t n, const double* states, const double* beta, const double* chi1,
                   const double* chi2, const double* kq1, const double* kq2, uint32_t terms,
                   const double* E0, const double* J0, int mode, int newton_iters, double newton_tol,
                   double* out, int32_t* ok) {
  const ParamArrays A = {beta, chi1, chi2, kq1, kq2, terms};
  if (precision == 0) correct_t<long double>(n, states, A, E0, J0, mode, newton_iters, newton_tol, out, ok);
  else correct_t<double>(n, states, A, E0, J0, mode, newton_iters, newton_tol, out, ok);
  return 0;
}

int oracle_integrate(int precision, int64_t n, const double* states, const double* beta, const double* chi1,
                     const double* chi2, const double* kq1, const double* kq2, uint32_t terms, double h,
                     int64_t n_steps, int mode, double shadow_eps, int renorm_interval, int newton_iters,
                     double newton_tol, double r_merge, double r_escape, double* out_states,
                     double* out_invariants, double* out_fli, int32_t* out_status, int64_t* out_step,
                     int64_t* out_gn_steps, int n_threads, int integrator, int64_t sample_interval,
                     double* out_samples, double* out_shadow, double* out_diss) {
  const ParamArrays A = {beta, chi1, chi2, kq1, kq2, terms};
  const Options O = {mode, renorm_interval, newton_iters, newton_tol, r_merge, r_escape, integrator};
  if (n_threads <= 0) n_threads = omp_get_max_threads();
  if (precision == 0)
    integrate_t<long double>(n, states, A, h, n_steps, shadow_eps, O, out_states, out_invariants, out_fli,
                             out_status, out_step, out_gn_steps, n_threads, sample_interval, out_samples, out_shadow, out_diss);
  else
    integrate_t<double>(n, states, A, h, n_steps, shadow_eps, O, out_states, out_invariants, out_fli,
                        out_status, out_step, out_gn_steps, n_threads, sample_interval, out_samples, out_shadow, out_diss);
  return 0;
}

// Exact flop counts of the oracle's own formulation on one orbit (add, sub, mul,
// div, sqrt = 1 each): counts[0] = rhs, [1] = rk4_step, [2] = correct(mode),
// [3] = hamiltonian, [4] = gradient.  The correction is counted with tolerance 0,
// i.e. with all newton_iters steps taken.
int oracle_count_flops(const double* state12, double beta, double chi1, double chi2, double kq1, double kq2,
                       uint32_t terms, int mode, int newton_iters, long long* counts) {
  const State<Counted> z = load_state<Counted>(state12, 1, 0);
  const Params<Counted> P = {Counted(beta), Counted(chi1), Counted(chi2), Counted(kq1), Counted(kq2), terms};
  const Refs<Counted> R = references(z, P);
  Counted::flops = 0; (void)rhs(z, P); counts[0] = Counted::flops;
  Counted::flops = 0; State<Counted> zn = rk4_step(z, Counted(1.0), P); counts[1] = Counted::flops;
  Counted::flops = 0; (void)correct(zn, P, R, mode, newton_iters, Counted(0.0)); counts[2] = Counted::flops;
  Counted::flops = 0; (void)hamiltonian(z, P); counts[3] = Counted::flops;
  Counted::flops = 0; (void)gradient(z, P); counts[4] = Counted::flops;
  return 0;
}

int oracle_max_threads(void) { return omp_get_max_threads(); }

}  // extern "C"
