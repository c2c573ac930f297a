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

enum { ST_OK = 0, ST_MERGED = 1, ST_UNBOUND = 2, ST_NONFINITE = 3, ST_NEWTON_FLAG = 256 };

// Status of a completed step from the main trajectory's |r|^2 (R13).  The non-finite
// test is integer work and stays with the caller.  Used by the kernel's step loop and by the flop model.
template <class T>
MC_DEV int radius_status(const T* z, T r_merge2, T r_escape2) {
  const T r2 = dot3(z, z);
  return (r2 < r_merge2) ? ST_MERGED : ((r2 > r_escape2) ? ST_UNBOUND : ST_OK);
}

// One shadow renormalisation (R10-R12): d = |y - ym| over all 12 components, FLI accumulator += log10(d / d0),
// the shadow y is pulled back onto the main state ym at distance d0 along y - ym, its spins are renormalised (eq 10) and
// its reference integrals re-taken from the new state (R11).  Returns false, leaving everything untouched, when d is
// zero or not finite.  Used by the kernel's step loop and by the flop model.
template <int MODE, bool QM, class C, class T>
MC_DEV bool renormalise_shadow(const C& c, T* y, const T* ym, T d0, T& acc, RefsT<T>& R) {
  T d2 = 0.0;
#pragma unroll
  for (int i = 0; i < 12; ++i) { const T e = y[i] - ym[i]; d2 = fma(e, e, d2); }
  const T d = sqrt_pos(d2);
  if (!(d > T(0.0)) || !(d < T(1.0e300))) return false;
  acc += log10_(div_exact(d, d0));
  const T s = div_exact(d0, d);
#pragma unroll
  for (int i = 0; i < 12; ++i) y[i] = fma(s, y[i] - ym[i], ym[i]);
  if (MODE >= 1) { normalise3(y + 6); normalise3(y + 9); }
  references<QM>(c, y, R);
  return true;
}

// Mode 3: minimal-norm Gauss-Newton projection of (r,p) onto {H = E0, r x p = Lt}, Lt = J0 - S1 - S2.
// Constraint Jacobian D (4 x 6): row (a, b) = (dH/dr, dH/dp) and the three rows (p x e_k, e_k x r) of r x p.  The
// step is d = D^T (D D^T)^-1 F, F = (H - E0, r x p - Lt), z <- z - d.  The oracle assembles D D^T and solves it by
// pivoted elimination.  Here the same step is written out in the frame {r, p, L = r x p}:
//   * the three L-rows have the null space N = span{n1 = (r, -p), n2 = (p, 0), n3 = (0, r)} (the deformations of
//     (r, p) that keep r x p) and the row space {(p x l, l x r)}.  d = x + y, x in the row space, y in N.
//   * x is fixed by the L-rows alone: M l = r x p - Lt, M = (r.r + p.p) I - r r^T - p p^T.  M maps r -> pp r - rp p,
//     p -> rr p - rp r, L -> (rr + pp) L, so with l = lr r + lp p + lL L:  lr = -(Lt.r)/LL, lp = -(Lt.p)/LL,
//     lL = (LL - Lt.L)/((rr + pp) LL), LL = |L|^2, and  p x l = -lr L + lL (pp r - rp p),  l x r = -lp L + lL (rr p - rp r).
//   * y = g_N (f0 - g.x)/|g_N|^2, g_N the projection of g = (a, b) on N: g_N = sum_i alpha_i n_i, G alpha = beta,
//     beta = (a.r - b.p, a.p, b.r), G = Gram matrix of n1..n3 = [[rr+pp, rp, -rp], [rp, pp, 0], [-rp, 0, rr]],
//     det G = (rr + pp) LL, |g_N|^2 = beta.alpha.
// So the step needs the gradient only through six dot products (with r, p, L), and those follow from the scalars of
// the model routine without ever forming a and b (dH/dr = w1 s1 + w2 s2 + Cr r + B p + p x Sg, dH/dp = A p + B r +
// Sg x r, Sg = u^3 (k1 sigma1 + k2 sigma2)):
//   a.r = w1 a1 + w2 a2 + Cr rr + B rp + H_SO      b.p = A pp + B rp + H_SO
//   a.p = w1 b1 + w2 b2 + Cr rp + B pp             b.r = A rp + B rr
//   a.L = w1 l1 + w2 l2 + rp (Sg.p) - pp (Sg.r)    b.L = rp (Sg.r) - rr (Sg.p)
// with a_i = sigma_i.r, b_i = sigma_i.p, l_i = sigma_i.L.  One reciprocal per step, no cross product besides L.
//
// gn_pass: ONE Gauss-Newton step on (r, p) = z[0:6] with the spins z[6:12] held fixed.  Returns whether another step
// is needed: |(dr,dp)|^2 > tol^2 p.p (R6); false also for a non-finite step.
template <bool QM, class C, class T>
MC_DEV bool gn_pass(const C& c, T* z, const T& E0, const T* Lt, double tol2) {
  T* r = z;
  T* p = z + 3;
  const T* s1 = z + 6;
  const T* s2 = z + 9;
  OrbitalScalars<T> o;
  orbital_scalars<true>(c, r, p, o);
  const T rr = o.r2, pp = o.P, rp = o.rp, A = o.A, B = o.B;
  T L[3];
  cross3(r, p, L);
  const T a1 = dot3(s1, r), a2 = dot3(s2, r);
  const T b1 = dot3(s1, p), b2 = dot3(s2, p);
  const T l1 = dot3(s1, L), l2 = dot3(s2, L);
  const T k1u = c[K_K1] * o.u3, k2u = c[K_K2] * o.u3;
  const T LS = fma(k2u, l2, k1u * l1);                 // H_SO = L.Sg
  const T Sgr = fma(k2u, a2, k1u * a1);                // Sg.r
  const T Sgp = fma(k2u, b2, k1u * b1);                // Sg.p
  SpinScalars<T> q;
  spin_scalars<QM, true>(c, s1, s2, o, a1, a2, o.u5 * a1, o.u5 * a2, LS, q);
  const T Cr = o.u2 * fma(3.0, q.X, -o.Cu);
  const T H = orbital_energy(c, o) + (LS + q.Hss);
  const T f0 = H - E0;
  // the gradient's six dot products
  const T t = fma(B, rp, LS);
  const T ar = fma(q.w1, a1, fma(q.w2, a2, fma(Cr, rr, t)));
  const T bp = fma(A, pp, t);
  const T ap = fma(q.w1, b1, fma(q.w2, b2, fma(Cr, rp, B * pp)));
  const T br = fma(A, rp, B * rr);
  const T aL = fma(q.w1, l1, fma(q.w2, l2, fma(rp, Sgp, -(pp * Sgr))));
  const T bL = fma(rp, Sgr, -(rr * Sgp));
  // x: the L-rows
  const T rp2 = rp * rp;
  const T LL = fma(rr, pp, -rp2);
  const T spp = rr + pp;
  const T D = spp * LL;                                 // det G
  const T mr = dot3(Lt, r), mp = dot3(Lt, p), nL = LL - dot3(Lt, L);   // lr = -mr/LL, lp = -mp/LL, lL = nL/D
  // D (g.x) = (rr + pp)(mr a.L + mp b.L) + nL (pp a.r - rp (a.p + b.r) + rr b.p)
  const T Dgx = fma(nL, fma(pp, ar, fma(rr, bp, -(rp * (ap + br)))), spp * fma(mr, aL, mp * bL));
  // y: D alpha = adj(G) beta, T = D |g_N|^2
  const T be1 = ar - bp;
  const T C12 = -(rp * rr), C13 = rp * pp;
  const T al1 = fma(rr * pp, be1, fma(C12, ap, C13 * br));
  const T al2 = fma(C12, be1, fma(fma(rr, rr, LL), ap, -(rp2 * br)));
  const T al3 = fma(C13, be1, fma(fma(pp, pp, LL), br, -(rp2 * ap)));
  const T Tn = fma(be1, al1, fma(ap, al2, br * al3));
  const T TD = Tn * D;
  const T inv = (TD != 0.0) ? rcp_nz(TD) : T(0.0);     // singular only for r || p or a circular orbit: zero step
  const T invD = Tn * inv;
  const T sy = fma(f0, D, -Dgx) * inv;                  // (f0 - g.x) / (D |g_N|^2)
  const T lL = nL * invD;
  const T iLL = spp * invD;                             // 1 / LL
  const T y1 = sy * al1, lLrp = lL * rp;
  const T crr = fma(lL, pp, y1), crp = fma(sy, al2, -lLrp), crL = mr * iLL;      // dr = crr r + crp p + crL L
  const T cpr = fma(sy, al3, -lLrp), cpp = fma(lL, rr, -y1), cpL = mp * iLL;     // dp = cpr r + cpp p + cpL L
  T dd = 0.0;
  T dr[3], dp[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    dr[i] = fma(crr, r[i], fma(crp, p[i], crL * L[i]));
    dp[i] = fma(cpr, r[i], fma(cpp, p[i], cpL * L[i]));
    dd = fma(dr[i], dr[i], fma(dp[i], dp[i], dd));
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) { r[i] -= dr[i]; p[i] -= dp[i]; }
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
