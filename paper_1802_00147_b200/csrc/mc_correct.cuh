// mc_correct.cuh -- manifold correction operators C_mode,
// applied in registers right after the RK4 step.
#pragma once
#include "mc_math.cuh"

namespace mc {

template <class T> struct RefsT { T E0, J0[3]; };   // reference integrals "at the starting time"
typedef RefsT<double> Refs;

#ifdef __CUDACC__
__device__ __forceinline__ bool warp_any(bool b) { return __any_sync(0xffffffffu, b); }
__device__ __forceinline__ double abs_(double x) { return fabs(x); }
#endif

template <bool QM, class C, class T>
MC_DEV void references(const C& c, const T* z, RefsT<T>& R) {
  R.E0 = hamiltonian<QM>(c, z);
  total_J(c, z, R.J0);
}

// Mode 3: minimal-norm Gauss-Newton projection of (r,p) onto {H = E0, r x p = J0 - S1 - S2}.
// Constraint Jacobian rows: (a, b) = (dH/dr, dH/dp) and (p x e_k, e_k x r).  D D^T is
//   [ g   c^T ]      g = a.a + b.b,  c = a x p + r x b,
//   [ c   M   ]      M = (r.r + p.p) I - r r^T - p p^T
// M^-1 is closed-form (Woodbury): M^-1 x = N(x)/D, D = (r.r + p.p) |L|^2,
//   N(x) = |L|^2 x + r (rr (r.x) + rp (p.x)) + p (rp (r.x) + pp (p.x)),
// so the 4x4 solve needs one reciprocal.  The oracle solves the same system by pivoted elimination.
//
// gn_pass: ONE Gauss-Newton step on (r, p) = z[0:6] with the spins z[6:12] held fixed, towards energy E0 and orbital
// angular momentum Lt = J0 - S1 - S2.  Returns whether another step is needed: |(dr,dp)|^2 > tol^2 p.p (R6;
// PAPER.md:146, 197); false also for a non-finite step.
template <bool QM, class C, class T>
MC_DEV bool gn_pass(const C& c, T* z, const T& E0, const T* Lt, double tol2) {
  T g[12], H;
  pn_eval<QM, false, true, false>(c, z, g, H);
  T* r = z;
  T* p = z + 3;
  const T* a = g;
  const T* b = g + 3;
  T fL[3], cv[3];
  cross3(r, p, fL);
#pragma unroll
  for (int i = 0; i < 3; ++i) fL[i] -= Lt[i];
  const T f0 = H - E0;
  // c = a x p + r x b
  cv[0] = fma(r[1], b[2], fma(-r[2], b[1], fma(a[1], p[2], -(a[2] * p[1]))));
  cv[1] = fma(r[2], b[0], fma(-r[0], b[2], fma(a[2], p[0], -(a[0] * p[2]))));
  cv[2] = fma(r[0], b[1], fma(-r[1], b[0], fma(a[0], p[1], -(a[1] * p[0]))));
  const T gg = dot3(a, a) + dot3(b, b);
  const T rr = dot3(r, r), pp = dot3(p, p), rp = dot3(r, p);
  const T LL = fma(rr, pp, -(rp * rp));
  const T D = (rr + pp) * LL;
  // N(c), N(fL)
  const T rc = dot3(r, cv), pc = dot3(p, cv), rf = dot3(r, fL), pf = dot3(p, fL);
  const T cr_ = fma(rp, pc, rr * rc), cp_ = fma(pp, pc, rp * rc);
  const T fr_ = fma(rp, pf, rr * rf), fp_ = fma(pp, pf, rp * rf);
  T Nc[3], Nf[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    Nc[i] = fma(p[i], cp_, fma(r[i], cr_, LL * cv[i]));
    Nf[i] = fma(p[i], fp_, fma(r[i], fr_, LL * fL[i]));
  }
  const T S = fma(gg, D, -dot3(cv, Nc));
  const T num = fma(D, f0, -dot3(cv, Nf));
  const T DS = D * S;
  const T inv = (DS != 0.0) ? rcp_nz(DS) : T(0.0);      // singular only for r || p or a circular orbit
  const T l0 = num * D * inv;                         // num / S
  const T sD = S * inv;                               // 1 / D
  T lL[3], d1[3], d2[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) lL[i] = fma(-l0, Nc[i], Nf[i]) * sD;
  cross3(p, lL, d1);   // dr = l0 a + p x lL
  cross3(lL, r, d2);   // dp = l0 b + lL x r
  T dd = 0.0;
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const T dr = fma(l0, a[i], d1[i]);
    const T dp = fma(l0, b[i], d2[i]);
    dd = fma(dr, dr, fma(dp, dp, dd));
    r[i] -= dr;
    p[i] -= dp;
  }
  return dd > tol2 * pp;
}

// Iteration control (R6): a lane repeats the step until its last update satisfies the test, at most `iters`
// times.  The decision is per lane (results do not depend on the neighbours); the warp leaves the loop when no lane
// needs another step.  Must be called by all 32 lanes.  Returns the number of steps this lane took; warp_passes
// receives the number of passes the WARP made through the loop body (= the largest step count among its lanes: what
// the pipe really executed).
template <bool QM, class C, class T>
MC_DEV int project_six(const C& c, T* z, const RefsT<T>& R, int iters, double tol2, int& warp_passes) {
  T Lt[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) Lt[i] = fma(-c[K_S2], z[9 + i], fma(-c[K_S1], z[6 + i], R.J0[i]));
  bool need = true;
  int done = 0;
  warp_passes = 0;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    if (!warp_any(need)) break;
    ++warp_passes;
    if (need) {
      need = gn_pass<QM>(c, z, R.E0, Lt, tol2);
      ++done;
    }
  }
  return done;
}

// Mode 2: the paper's dual scaling p <- alpha p*, r <- beta_s r* (eq 11) solving H = E0, |J| = |J0|
// (eqs 12-13 at their exact root, R5).  With v = 1/beta_s, gamma = alpha beta_s every term of
// H is a monomial in (alpha, v), so g(v) = H(gamma v, v) - E0 is a degree-6 polynomial whose
// coefficients are computed once; gamma is the root of the |J| quadratic.  Returns false if skipped.
template <bool QM, class C, class T>
MC_DEV bool dual_scaling(const C& c, T* z, const RefsT<T>& R, int iters, double tol) {
  const T* r = z;
  const T* p = z + 3;
  const T* s1 = z + 6;
  const T* s2 = z + 9;
  T L[3], S[3];
  cross3(r, p, L);
#pragma unroll
  for (int i = 0; i < 3; ++i) S[i] = fma(c[K_S2], s2[i], c[K_S1] * s1[i]);
  const T LL = dot3(L, L), LS = dot3(L, S), SS = dot3(S, S), J02 = dot3(R.J0, R.J0);
  const T disc = fma(LS, LS, -(LL * (SS - J02)));
  if (!(disc >= 0.0) || !(LL > 0.0)) return false;
  const T sg = (LL + LS >= 0.0) ? T(1.0) : T(-1.0);
  const T gam = div_(sg * sqrt_pos(disc) - LS, LL);
  // starred scalars
  const T u = rsqrt_pos(dot3(r, r));
  const T u2 = u * u, u3 = u2 * u, u5 = u3 * u2;
  const T rp = dot3(r, p), P = dot3(p, p);
  const T npu = rp * u, Q = npu * npu;
  const T a1 = dot3(s1, r), a2 = dot3(s2, r), d12 = dot3(s1, s2);
  T Sg[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) Sg[i] = fma(c[K_K2], s2[i], c[K_K1] * s1[i]);
  const T Hso = u3 * dot3(L, Sg);
  T Hss = c[K_C12] * fma(3.0 * a1 * a2, u5, -(d12 * u3));
  if (QM) {
    Hss += c[K_Q1] * fma(3.0 * a1 * a1, u5, -(dot3(s1, s1) * u3));
    Hss += c[K_Q2] * fma(3.0 * a2 * a2, u5, -(dot3(s2, s2) * u3));
  }
  const T g2 = gam * gam, g4 = g2 * g2, g6 = g4 * g2;
  // g(v) = -E0 + k1 v + k2 v^2 + ... + k6 v^6
  const T k1 = -u;
  const T k2 = fma(0.5 * g2, P, c[K_H1] * u2);
  const T k3 = fma(g2 * u, fma(c[K_B1], P, c[K_B2] * Q), fma(c[K_F1], u3, fma(gam, Hso, Hss)));
  const T k4 = fma(g4 * c[K_A1], P * P, g2 * u2 * fma(c[K_E1], P, c[K_E2] * Q));
  const T k5 = g4 * u * fma(P, fma(c[K_D1], P, c[K_D2] * Q), c[K_D3] * Q * Q);
  const T k6 = g6 * c[K_C3] * P * P * P;
  T v = 1.0, dv = 0.0;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
    const T gv = fma(v, fma(v, fma(v, fma(v, fma(v, fma(v, k6, k5), k4), k3), k2), k1), -R.E0);
    const T dg = fma(v, fma(v, fma(v, fma(v, fma(v, 6.0 * k6, 5.0 * k5), 4.0 * k4), 3.0 * k3), 2.0 * k2), k1);
    dv = -div_(gv, dg);
    v += dv;
  }
  if (!is_finite(v) || !(abs_(dv) <= tol) || !(abs_(v - 1.0) <= 1e-3)) return false;
  const T bs = div_(T(1.0), v), al = gam * v;
#pragma unroll
  for (int i = 0; i < 3; ++i) { z[i] *= bs; z[3 + i] *= al; }
  return true;
}

// C_mode: spins first (eq 10), then (r,p) with the corrected spins.
// gn_steps receives the number of Gauss-Newton steps mode 3 took (0 otherwise), warp_passes the passes of the warp.
template <int MODE, bool QM, class C, class T>
MC_DEV bool correct(const C& c, T* z, const RefsT<T>& R, int iters, double tol, int& gn_steps, int& warp_passes);
template <int MODE, bool QM, class C, class T>
MC_DEV bool correct(const C& c, T* z, const RefsT<T>& R, int iters, double tol, int& gn_steps) {
  int wp;
  return correct<MODE, QM>(c, z, R, iters, tol, gn_steps, wp);
}
template <int MODE, bool QM, class C, class T>
MC_DEV bool correct(const C& c, T* z, const RefsT<T>& R, int iters, double tol, int& gn_steps, int& warp_passes) {
  gn_steps = 0;
  warp_passes = 0;
  if (MODE >= 1) { normalise3(z + 6); normalise3(z + 9); }
  if (MODE == 2) return dual_scaling<QM>(c, z, R, iters, tol);
  if (MODE == 3) gn_steps = project_six<QM>(c, z, R, iters, tol * tol, warp_passes);
  return true;
}

}  // namespace mc
