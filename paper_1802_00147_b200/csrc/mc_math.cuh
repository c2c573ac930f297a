// mc_math.cuh -- per-trajectory math: fused Hamiltonian / gradient / precession routine, classical RK4,
// Butcher RK5.  Everything lives in registers; one thread = one trajectory.
//
// Formulation: unit spins, raw dot products (no unit vector n), all inverse
// powers of r from one rsqrt, Horner polynomials in P = p.p, Q = (n.p)^2, u = 1/r, FMA-first.
// The oracle (oracle/pn_oracle.hpp) is written differently on purpose; the two share no code.
//
// Every routine is a template on the scalar type T.  The kernels use T = double.  The host-only flop model
// (mc_flop_model.cpp, plain C++) instantiates the very same routines with T = mc::Cnt, a scalar that counts
// its own FMAs, multiplications, additions and special functions -- so the algorithmic flop figures bench.py
// reports are derived from the code that runs, not from a hand count.
#pragma once
#include "mc_consts.h"

#ifdef __CUDACC__
#define MC_DEV __device__ __forceinline__
#else
#include <cmath>
#define MC_DEV inline
#endif

namespace mc {

// ---- constant providers -------------------------------------------------------------------------
// Uniform parameters: the struct is a __grid_constant__ kernel parameter, so c[i] is a constant-bank
// operand of the DFMA itself (no register, no load).  Per-orbit parameters: one slot per thread in
// shared memory, laid out [MC_NCONST][blockDim.x] (conflict-free LDS.64).
struct UniformConsts {
  const McConsts& k;
  MC_DEV double operator[](int i) const { return k.v[i]; }
};
struct SharedConsts {
  const double* base;  // &smem[threadIdx.x]
  int stride;          // blockDim.x
  MC_DEV double operator[](int i) const { return base[i * stride]; }
};
// Uniform beta, chi1, chi2 with per-orbit quadrupole coefficients kappa_i (BASELINE config 3; mc_params.per_orbit
// = 2): the constants that do not depend on kappa stay constant-bank operands, the four that do (q_i, 3 m_ii;
// all linear in kappa_i) ride in registers.  i is a compile-time constant wherever this is called, so the
// selection folds away.
struct KappaConsts {
  const McConsts& k;   // derived with kappa = 1
  double q1, q2, m11x3, m22x3;
  MC_DEV double operator[](int i) const {
    return i == K_Q1 ? q1 : (i == K_Q2 ? q2 : (i == K_3M11 ? m11x3 : (i == K_3M22 ? m22x3 : k.v[i])));
  }
};

#ifdef __CUDACC__
// 1/sqrt(x) for x > 0, normal: MUFU.RSQ64H seed (~2^-22 relative) + one third-order step
// y <- y (1 + e/2 + 3 e^2/8), e = 1 - x y^2  => relative error ~ 1e-20 before rounding.
__device__ __forceinline__ double rsqrt_pos(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);
  const double q = fma(0.375, e, 0.5) * e;
  return fma(y, q, y);
}

// 1/x for finite normal x != 0: MUFU.RCP64H seed + two Newton steps.
__device__ __forceinline__ double rcp_nz(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, fma(e, e, e), y);   // y (1 + e + e^2): error e^3
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}
__device__ __forceinline__ double sqrt_pos(double x) { return sqrt(x); }
// a / b for mode 2's quadratic root and Newton updates: a times the refined reciprocal (<= 1.5 ulp; no IEEE division
// sequence with its slow path in the step loop).  b = 0 or non-finite gives a non-finite result, which the caller's
// skip test catches just as it would after a true division.
__device__ __forceinline__ double div_(double a, double b) { return a * rcp_nz(b); }
// IEEE division and log10 for the shadow renormalisation (once per renorm_interval steps, outside the hot sequence)
__device__ __forceinline__ double div_exact(double a, double b) { return a / b; }
__device__ __forceinline__ double log10_(double x) { return log10(x); }
__device__ __forceinline__ bool is_finite(double v) { return (((unsigned)__double2hiint(v)) & 0x7ff00000u) != 0x7ff00000u; }

__device__ __forceinline__ bool finite12(const double* z) {
  // exponent field all ones <=> inf or nan <=> (high word with the sign shifted out) >= 0xffe00000.  Integer pipe
  // only (keeps the FP64 pipe for the physics); a max tree, not a predicate chain, so the dependency depth is 4.
  unsigned m[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) m[i] = (unsigned)__double2hiint(z[i]) << 1;
  const unsigned a = max(max(m[0], m[1]), m[2]), b = max(max(m[3], m[4]), m[5]);
  const unsigned c = max(max(m[6], m[7]), m[8]), d = max(max(m[9], m[10]), m[11]);
  return max(max(a, b), max(c, d)) < 0xffe00000u;
}
#endif

// ---- small helpers ------------------------------------------------------------------------------
template <class T>
MC_DEV T dot3(const T* a, const T* b) {
  return fma(a[2], b[2], fma(a[1], b[1], a[0] * b[0]));
}
// c = a x b
template <class T>
MC_DEV void cross3(const T* a, const T* b, T* c) {
  c[0] = fma(a[1], b[2], -(a[2] * b[1]));
  c[1] = fma(a[2], b[0], -(a[0] * b[2]));
  c[2] = fma(a[0], b[1], -(a[1] * b[0]));
}

// ---- the fused model routine ----------------------------------------------------------------------
// Scalars of the orbital part (N + 1PN + 2PN) at one point: everything is a polynomial in P = p.p, Q = (n.p)^2 and
// u = 1/|r| (Horner; every constant multiple is precomputed, mc_consts.h).
//   dH_orb/dp = A p + B r,   dH_orb/dr = B p - u^2 Cu r
template <class T>
struct OrbitalScalars { T r2, u, u2, u3, u5, rp, P, w, Q, t1, t2, t3, A, B, Cu; };

template <bool WANT_H, class C, class T>
MC_DEV void orbital_scalars(const C& c, const T* r, const T* p, OrbitalScalars<T>& o) {
  o.r2 = dot3(r, r);
  o.u = rsqrt_pos(o.r2);
  o.u2 = o.u * o.u; o.u3 = o.u2 * o.u; o.u5 = o.u3 * o.u2;
  o.rp = dot3(r, p);
  o.P = dot3(p, p);
  o.w = o.rp * o.u2;                                          // (n.p) u
  o.Q = o.rp * o.w;                                           // (n.p)^2
  const T u = o.u, P = o.P, Q = o.Q;
  o.t1 = fma(c[K_D2], Q, fma(c[K_D1], P, c[K_B1]));           // b1 + d1 P + d2 Q
  o.t2 = fma(c[K_D3], Q, c[K_B2]);                            // b2 + d3 Q
  o.t3 = WANT_H ? fma(c[K_E2], Q, c[K_E1] * P) : T(0.0);      // e1 P + e2 Q (only H itself needs it)
  // H_P = 1/2 + P (2 a1 + 3 c3 P) + u (b1 + 2 d1 P + d2 Q + e1 u)
  const T hp_u = fma(c[K_E1], u, fma(c[K_D1], P, o.t1));
  const T HP = fma(u, hp_u, fma(P, fma(c[K_3C3], P, c[K_2A1]), 0.5));
  // 2 H_Q = u (2 b2 + 2 d2 P + 4 d3 Q + 2 e2 u)
  const T HQ2 = u * fma(c[K_4D3], Q, fma(c[K_2D2], P, fma(c[K_2E2], u, c[K_2B2])));
  // H_u = -1 + P t1 + Q t2 + u (2 h1 + 2 t3 + 3 f1 u)
  const T hu_u = WANT_H ? fma(c[K_3F1], u, fma(2.0, o.t3, c[K_2H1]))
                        : fma(c[K_3F1], u, fma(c[K_2E1], P, fma(c[K_2E2], Q, c[K_2H1])));
  const T Hu = fma(u, hu_u, fma(Q, o.t2, fma(P, o.t1, -1.0)));
  o.A = HP + HP;
  o.B = HQ2 * o.w;
  o.Cu = fma(Hu, u, HQ2 * Q);
}

// H_orb = P/2 - u + P^2 (a1 + c3 P) + u (P t1 + Q t2) + u^2 (h1 + t3) + f1 u^3
template <class C, class T>
MC_DEV T orbital_energy(const C& c, const OrbitalScalars<T>& o) {
  return fma(o.u2, fma(c[K_F1], o.u, c[K_H1] + o.t3),
             fma(o.u, fma(o.Q, o.t2, o.P * o.t1), fma(o.P * o.P, fma(c[K_C3], o.P, c[K_A1]), fma(0.5, o.P, -o.u))));
}

// Spin-spin (and quadrupole-monopole) scalars from a_i = sigma_i.r, d_ij = sigma_i.sigma_j and LS = H_SO:
//   X:  the coefficient of r in dH_spin/dr is 3 u^2 X,  X = -H_SO + c12 (d12 u^3 - 5 a1 a2 u^5) + QM
//   w_i: the coefficient of sigma_i in dH_spin/dr;  Hss = H_12 + H_11 + H_22 (WANT_H)
template <class T>
struct SpinScalars { T X, w1, w2, Hss; };

template <bool QM, bool WANT_H, class C, class T>
MC_DEV void spin_scalars(const C& c, const T* s1, const T* s2, const OrbitalScalars<T>& o, const T& a1, const T& a2,
                         const T& ua1, const T& ua2 /* u^5 a_i */, const T& LS, SpinScalars<T>& q) {
  const T d12 = dot3(s1, s2);
  const T a12u5 = a1 * ua2;
  const T c12u3 = c[K_C12] * o.u3;
  q.X = fma(c12u3, d12, fma(c[K_M5C12], a12u5, -LS));
  q.w1 = c[K_3C12] * ua2;
  q.w2 = c[K_3C12] * ua1;
  q.Hss = fma(c[K_3C12], a12u5, -(c12u3 * d12));
  if (QM) {
    // H_ii = q_i (3 a_i^2 u^5 - d_ii u^3).  Only q_i itself is used as a constant (no multiples), so that the
    // per-orbit-kappa variant keeps one register per body; the numeric factors ride as FMA immediates.
    const T d11 = dot3(s1, s1), d22 = dot3(s2, s2);
    const T q1u3 = c[K_Q1] * o.u3, q2u3 = c[K_Q2] * o.u3;
    const T q1a = c[K_Q1] * ua1, q2a = c[K_Q2] * ua2;          // q_i u^5 a_i
    const T q1aa = q1a * a1, q2aa = q2a * a2;                  // q_i u^5 a_i^2
    q.X = fma(q1u3, d11, fma(-5.0, q1aa, q.X));
    q.X = fma(q2u3, d22, fma(-5.0, q2aa, q.X));
    q.w1 = fma(6.0, q1a, q.w1);
    q.w2 = fma(6.0, q2a, q.w2);
    if (WANT_H) q.Hss += fma(3.0, q1aa, -(q1u3 * d11)) + fma(3.0, q2aa, -(q2u3 * d22));
  }
}

// Input  z = (r[0:3], p[3:6], sigma1[6:9], sigma2[9:12]).
// Output g[0:3] = dH/dr, g[3:6] = dH/dp; if OMEGA: g[6:9] = Omega1, g[9:12] = Omega2; if WANT_H: H.
// With RR (2.5PN radiation reaction, MC_TERM_RR; only the equations of motion use it): g[0:3] = dH/dr - F, so that
// dp/dt = -g as in the conservative case, and g[12] = (dH/dp).F, g[13:16] = r x F, the rates of the work and torque
// integrals W, G.  F = fr r + fp p has no other components, so it costs two coefficients:
// r x F = fp L, v.F = fr (v.r) + fp (v.p) with v.r = A (r.p) + B r^2, v.p = A P + B (r.p) + H_SO.
// eqs (1)-(9) of the paper with the readings of DESIGN.md section 3.
template <bool QM, bool OMEGA, bool WANT_H, bool RR, class C, class T>
MC_DEV void pn_eval(const C& c, const T* z, T* g, T& H) {
  const T* r = z;
  const T* p = z + 3;
  const T* s1 = z + 6;
  const T* s2 = z + 9;
  OrbitalScalars<T> o;
  orbital_scalars<WANT_H>(c, r, p, o);
  const T u2 = o.u2, u3 = o.u3, u5 = o.u5, A = o.A, B = o.B;

  // spin couplings
  const T a1 = dot3(s1, r), a2 = dot3(s2, r);
  const T ua1 = u5 * a1, ua2 = u5 * a2;                               // every a_i that meets u^5 does so through these
  const T k1u = c[K_K1] * u3, k2u = c[K_K2] * u3;
  T Sg[3], L[3], SxR[3], PxS[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) Sg[i] = fma(k2u, s2[i], k1u * s1[i]);   // u^3 (k1 sigma1 + k2 sigma2)
  cross3(r, p, L);
  cross3(Sg, r, SxR);
  cross3(p, Sg, PxS);
  const T LS = dot3(L, Sg);                                      // = H_SO
  SpinScalars<T> q;
  spin_scalars<QM, WANT_H>(c, s1, s2, o, a1, a2, ua1, ua2, LS, q);
  T Cr = u2 * fma(3.0, q.X, -o.Cu);                   // coefficient of r in dH/dr
  T Bp = B;                                           // coefficient of p in dH/dr
  if constexpr (RR) {
    const T ca = fma(c[K_RA3], o.Q, fma(c[K_RA2], o.u, c[K_RA1] * o.P));
    const T cb = fma(c[K_RB3], o.Q, fma(c[K_RB2], o.u, c[K_RB1] * o.P));
    const T fr = ca * o.w * u3, fp = -(cb * u3);       // F = fr r + fp p
    Cr -= fr;
    Bp -= fp;
    g[12] = fma(fr, fma(A, o.rp, B * o.r2), fp * fma(A, o.P, fma(B, o.rp, LS)));
#pragma unroll
    for (int i = 0; i < 3; ++i) g[13 + i] = fp * L[i];
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    g[i] = fma(q.w2, s2[i], fma(q.w1, s1[i], fma(Cr, r[i], fma(Bp, p[i], PxS[i]))));
    g[3 + i] = fma(A, p[i], fma(B, r[i], SxR[i]));
  }
  if (OMEGA) {
    const T o1u = c[K_O1] * u3, o2u = c[K_O2] * u3;
    const T m12u = c[K_M12] * u3, m21u = c[K_M21] * u3;
    T b1r = c[K_3M12] * ua2, b2r = c[K_3M21] * ua1;             // 3 u^5 (m12 a2 + m11 a1), 3 u^5 (m21 a1 + m22 a2)
    if (QM) { b1r = fma(c[K_3M11], ua1, b1r); b2r = fma(c[K_3M22], ua2, b2r); }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      g[6 + i] = fma(-m12u, s2[i], fma(b1r, r[i], o1u * L[i]));
      g[9 + i] = fma(-m21u, s1[i], fma(b2r, r[i], o2u * L[i]));
    }
  }
  if (WANT_H) H = orbital_energy(c, o) + (LS + q.Hss);
}

// dz/dt, eqs (6)-(7): dr/dt = dH/dp, dp/dt = -dH/dr (+ a_2.5PN), dsigma_i/dt = Omega_i x sigma_i.
// RR: 16 components, f[12] = dW/dt, f[13:16] = dG/dt.
template <bool QM, bool RR, class C, class T>
MC_DEV void pn_rhs(const C& c, const T* z, T* f) {
  T g[RR ? 16 : 12], H;
  pn_eval<QM, true, false, RR>(c, z, g, H);
#pragma unroll
  for (int i = 0; i < 3; ++i) { f[i] = g[3 + i]; f[3 + i] = -g[i]; }
  cross3(g + 6, z + 6, f + 6);
  cross3(g + 9, z + 9, f + 9);
  if constexpr (RR) {
#pragma unroll
    for (int i = 12; i < 16; ++i) f[i] = g[i];
  }
}

// J = r x p + s1 sigma1 + s2 sigma2
template <class C, class T>
MC_DEV void total_J(const C& c, const T* z, T* J) {
  cross3(z, z + 3, J);
#pragma unroll
  for (int i = 0; i < 3; ++i) J[i] = fma(c[K_S2], z[9 + i], fma(c[K_S1], z[6 + i], J[i]));
}

template <bool QM, class C, class T>
MC_DEV T hamiltonian(const C& c, const T* z) {
  T g[12], H;
  pn_eval<QM, false, true, false>(c, z, g, H);
  return H;
}

// Step weights: h times the coefficients of the two tableaus, formed once on the host (mc_api.cu) and carried in the
// kernel parameter.  The stage inputs y + (h c) k and the running sum of b_i k_i are 84 FMAs per RK4 step; with the
// weight in the constant bank each reads two registers (2 cycles on the FP64 pipe), with the weight in a register
// three (3 cycles, operand bandwidth).  The products are the ones the step routines used to
// form themselves in double precision, so results do not change by a bit.
enum McStepWeightIndex {
  HW_H = 0, HW_H2, HW_H3, HW_H6,                                                        // RK4: h, h/2, h/3, h/6
  HW_H790, HW_H3290, HW_H1290, HW_H4, HW_H8, HW_HM2, HW_H37, HW_H27, HW_H127, HW_H316, HW_H916, HW_H87   // RK5
};
struct StepWeights { double v[16]; };
MC_HD StepWeights step_weights(double h) {
  StepWeights w;
  w.v[HW_H] = h; w.v[HW_H2] = 0.5 * h; w.v[HW_H3] = h * (1.0 / 3.0); w.v[HW_H6] = h * (1.0 / 6.0);
  w.v[HW_H790] = h * (7.0 / 90.0); w.v[HW_H3290] = h * (32.0 / 90.0); w.v[HW_H1290] = h * (12.0 / 90.0);
  w.v[HW_H4] = 0.25 * h; w.v[HW_H8] = 0.125 * h; w.v[HW_HM2] = -0.5 * h;
  w.v[HW_H37] = h * (-3.0 / 7.0); w.v[HW_H27] = h * (2.0 / 7.0); w.v[HW_H127] = h * (12.0 / 7.0);
  w.v[HW_H316] = h * (3.0 / 16.0); w.v[HW_H916] = h * (9.0 / 16.0); w.v[HW_H87] = h * (8.0 / 7.0);
  return w;
}

// Classical RK4 (R9), low-storage bookkeeping: y (kept), acc, stage input yt.
// RR: components 12-15 (W, G) never enter the right-hand side, so they need no stage inputs: only their weighted
// sum of stage derivatives is accumulated.
template <bool QM, bool RR, class C, class T>
MC_DEV void rk4_step(const C& c, const T* y, const StepWeights& w, T* out) {
  constexpr int NS = RR ? 16 : 12;
  T k[NS], yt[12];
  pn_rhs<QM, RR>(c, y, k);
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H6], k[i], y[i]);
#pragma unroll
  for (int i = 0; i < 12; ++i) yt[i] = fma(w.v[HW_H2], k[i], y[i]);
  pn_rhs<QM, RR>(c, yt, k);
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H3], k[i], out[i]);
#pragma unroll
  for (int i = 0; i < 12; ++i) yt[i] = fma(w.v[HW_H2], k[i], y[i]);
  pn_rhs<QM, RR>(c, yt, k);
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H3], k[i], out[i]);
#pragma unroll
  for (int i = 0; i < 12; ++i) yt[i] = fma(w.v[HW_H], k[i], y[i]);
  pn_rhs<QM, RR>(c, yt, k);
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H6], k[i], out[i]);
}

// Butcher's six-stage fifth-order method (the paper's "RK5", R9):
//   c = 0, 1/4, 1/4, 1/2, 3/4, 1;  b = 7/90, 0, 32/90, 12/90, 32/90, 7/90
//   a2 = (1/4); a3 = (1/8, 1/8); a4 = (0, -1/2, 1); a5 = (3/16, 0, 0, 9/16); a6 = (-3/7, 2/7, 12/7, -12/7, 8/7)
// Bookkeeping: the linear combinations needed later (stage-4 input, stage-6 input, final sum) are accumulated as
// the stages arrive, so at most five 12-vectors are live besides the derivative being computed.  RR: components
// 12-15 only accumulate the final sum (see rk4_step).
template <bool QM, bool RR, class C, class T>
MC_DEV void rk5_step(const C& c, const T* y, const StepWeights& w, T* out) {
  constexpr int NS = RR ? 16 : 12;
  T k[NS], k1[12], yt[12], A4[12], S6[12];
  pn_rhs<QM, RR>(c, y, k);
#pragma unroll
  for (int i = 0; i < 12; ++i) { k1[i] = k[i]; yt[i] = fma(w.v[HW_H4], k[i], y[i]); }
#pragma unroll
  for (int i = 12; i < NS; ++i) out[i] = fma(w.v[HW_H790], k[i], y[i]);
  pn_rhs<QM, RR>(c, yt, k);                                                    // k2 (b2 = 0)
#pragma unroll
  for (int i = 0; i < 12; ++i) {
    yt[i] = fma(w.v[HW_H8], k[i], fma(w.v[HW_H8], k1[i], y[i]));
    A4[i] = fma(w.v[HW_HM2], k[i], y[i]);
    S6[i] = fma(w.v[HW_H27], k[i], fma(w.v[HW_H37], k1[i], y[i]));
  }
  pn_rhs<QM, RR>(c, yt, k);                                                    // k3
#pragma unroll
  for (int i = 0; i < 12; ++i) {
    yt[i] = fma(w.v[HW_H], k[i], A4[i]);
    S6[i] = fma(w.v[HW_H127], k[i], S6[i]);
    out[i] = fma(w.v[HW_H3290], k[i], fma(w.v[HW_H790], k1[i], y[i]));
  }
#pragma unroll
  for (int i = 12; i < NS; ++i) out[i] = fma(w.v[HW_H3290], k[i], out[i]);
  pn_rhs<QM, RR>(c, yt, k);                                                    // k4
#pragma unroll
  for (int i = 0; i < 12; ++i) {
    yt[i] = fma(w.v[HW_H916], k[i], fma(w.v[HW_H316], k1[i], y[i]));
    S6[i] = fma(-w.v[HW_H127], k[i], S6[i]);
  }
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H1290], k[i], out[i]);
  pn_rhs<QM, RR>(c, yt, k);                                                    // k5
#pragma unroll
  for (int i = 0; i < 12; ++i) yt[i] = fma(w.v[HW_H87], k[i], S6[i]);
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H3290], k[i], out[i]);
  pn_rhs<QM, RR>(c, yt, k);                                                    // k6
#pragma unroll
  for (int i = 0; i < NS; ++i) out[i] = fma(w.v[HW_H790], k[i], out[i]);
}

// INTEG: 0 classical RK4, 1 Butcher RK5
template <int INTEG, bool QM, bool RR, class C, class T>
MC_DEV void base_step(const C& c, const T* y, const StepWeights& w, T* out) {
  if (INTEG == 1) rk5_step<QM, RR>(c, y, w, out);
  else rk4_step<QM, RR>(c, y, w, out);
}

// eq (10): sigma <- sigma / |sigma|
template <class T>
MC_DEV void normalise3(T* s) {
  const T w = rsqrt_pos(dot3(s, s));
  s[0] *= w; s[1] *= w; s[2] *= w;
}

}  // namespace mc
