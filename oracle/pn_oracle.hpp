// pn_oracle.hpp -- CPU ORACLE (test infrastructure, NOT the product).
//
// Plain, slow, step-by-step restatement of the method of arXiv 1802.00147
// ("GPU accelerated manifold correction method for spinning compact binaries")
// as read in DESIGN.md: conservative PN Hamiltonian of a spinning binary,
// classical RK4, manifold correction onto the six integrals, two-nearby-
// trajectory FLI.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference leg may use anything under oracle/.
// It shares no code with paper_1802_00147_b200/ (the CUDA path): different
// variables (physical spins S_i, unit vector n, 1/r), gradients written term by
// term from the Hamiltonian, a generic pivoted 4x4 solver, no factoring.
//
// Everything is a template on the scalar type T: `long double` is the parity
// oracle, `double` is the timed CPU baseline (the paper's CPU code ran in
// double), `Counted` (pn_oracle_capi.cpp) counts flops.
//
// Units and symbols: G = c = M = 1; r in M, p in mu, H in mu,
// beta = m1/m2 <= 1, eta = mu/M = beta/(1+beta)^2, n = r/|r|.
// State z = (r, p, S1hat, S2hat): unit spins (eq 10); the spin
// vectors are S_i = s_i * S_i_hat with s1 = chi1*beta, s2 = chi2/beta, i.e.
// chi_i m_i^2 in units of mu*M (reading R2).
//
// Pins for every function in this file: tests/test_oracle_*.py (see the table
// in DESIGN.md section "Oracle pins"; a 480-mutant run over this file is
// recorded there).
// Parity unpinned (readings PAPER.md cannot fix, shared by both sides, listed in
// DESIGN.md section 6.3): the gauge (A, B) of the 2.5PN force in rr_force (R21:
// the paper does not print the expression; every gauge-invariant consequence is
// pinned), the unweighted 12-component norm of the FLI distance (R12), the
// identity metric of the mode-3 projection (R14), and the regular / chaotic
// labels the paper prints for its own orbits (R19 note).
#pragma once
#include <cmath>
#include <cstdint>

namespace pn_oracle {

// ---- scalar helpers (overloaded for Counted in the C API file) -------------
inline long double o_sqrt(long double x) { return sqrtl(x); }
inline double o_sqrt(double x) { return sqrt(x); }
inline long double o_log10(long double x) { return log10l(x); }
inline double o_log10(double x) { return log10(x); }
inline long double o_abs(long double x) { return fabsl(x); }
inline double o_abs(double x) { return fabs(x); }
inline bool o_finite(long double x) { return std::isfinite(x); }
inline bool o_finite(double x) { return std::isfinite(x); }

template <class T> struct V3 { T x, y, z; };
template <class T> inline V3<T> operator+(V3<T> a, V3<T> b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
template <class T> inline V3<T> operator-(V3<T> a, V3<T> b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
template <class T> inline V3<T> operator*(T s, V3<T> a) { return {s * a.x, s * a.y, s * a.z}; }
template <class T> inline T dot(V3<T> a, V3<T> b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
template <class T> inline V3<T> cross(V3<T> a, V3<T> b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}

// State of one trajectory: z = (r, p, S1hat, S2hat).
// Diss: with the 2.5PN radiation reaction (TERM_RR) the integrator also carries the work W = int (dr/dt).F dt and the
// torque integral G = int r x F dt of the dissipative force (the "integral invariant relation" of PAPER.md:221:
// H(t) - W(t) and J(t) - G(t) stay constant along the exact flow).  They are integrated by the same RK scheme as
// extra components; without TERM_RR their derivatives are zero and they never touch z.
template <class T> struct Diss { T w; V3<T> g; };
template <class T> struct State { V3<T> r, p, s1, s2; Diss<T> d; };
template <class T> inline Diss<T> operator+(Diss<T> a, Diss<T> b) { return {a.w + b.w, a.g + b.g}; }
template <class T> inline Diss<T> operator-(Diss<T> a, Diss<T> b) { return {a.w - b.w, a.g - b.g}; }
template <class T> inline Diss<T> operator*(T s, Diss<T> a) { return {s * a.w, s * a.g}; }
template <class T> inline State<T> operator+(State<T> a, State<T> b) {
  return {a.r + b.r, a.p + b.p, a.s1 + b.s1, a.s2 + b.s2, a.d + b.d};
}
template <class T> inline State<T> operator-(State<T> a, State<T> b) {
  return {a.r - b.r, a.p - b.p, a.s1 - b.s1, a.s2 - b.s2, a.d - b.d};
}
template <class T> inline State<T> operator*(T s, State<T> a) { return {s * a.r, s * a.p, s * a.s1, s * a.s2, s * a.d}; }
template <class T> inline T norm12sq(State<T> a) { return dot(a.r, a.r) + dot(a.p, a.p) + dot(a.s1, a.s1) + dot(a.s2, a.s2); }

enum : uint32_t { TERM_1PN = 1u, TERM_2PN = 2u, TERM_SO = 4u, TERM_S1S2 = 8u, TERM_QM = 16u, TERM_RR = 32u };

// Dynamic parameters of one binary (kq = quadrupole
// coefficient of DESIGN.md reading R16, kq = 1 for black holes).
template <class T> struct Params {
  T beta, chi1, chi2, kq1, kq2;
  uint32_t terms;
  T eta() const { return beta / ((T(1) + beta) * (T(1) + beta)); }
  T s1() const { return chi1 * beta; }   // |S1| in units of mu*M
  T s2() const { return chi2 / beta; }   // |S2| in units of mu*M
  T g1() const { return T(2) + T(3) / (T(2) * beta); }   // eq 8, coefficient of L
  T g2() const { return T(2) + T(3) * beta / T(2); }     // eq 9, coefficient of L
};

// ---- Hamiltonian, eq (1) without 3PN and 2.5PN -------------------------------
// H_N, H_1PN, H_2PN: ADM reduced two-body Hamiltonian (PAPER.md:86 points to
// Buonanno et al. 2006; R1).  H_SO: eta (L . (g1 S1 + g2 S2))/r^3
// (the L-terms of eqs 8-9).  H_S1S2, H_S1S1, H_S2S2: eqs (3)-(5) times eta.
template <class T> T hamiltonian(const State<T>& z, const Params<T>& P) {
  const T eta = P.eta();
  const T r = o_sqrt(dot(z.r, z.r));
  const V3<T> n = (T(1) / r) * z.r;
  const T p2 = dot(z.p, z.p);
  const T np = dot(n, z.p);
  T H = p2 / T(2) - T(1) / r;  // H_N
  if (P.terms & TERM_1PN) {
    H = H + (T(3) * eta - T(1)) / T(8) * p2 * p2
          - ((T(3) + eta) * p2 + eta * np * np) / (T(2) * r)
          + T(1) / (T(2) * r * r);
  }
  if (P.terms & TERM_2PN) {
    H = H + (T(1) - T(5) * eta + T(5) * eta * eta) / T(16) * p2 * p2 * p2
          + ((T(5) - T(20) * eta - T(3) * eta * eta) * p2 * p2
             - T(2) * eta * eta * np * np * p2
             - T(3) * eta * eta * np * np * np * np) / (T(8) * r)
          + ((T(5) + T(8) * eta) * p2 + T(3) * eta * np * np) / (T(2) * r * r)
          - (T(1) + T(3) * eta) / (T(4) * r * r * r);
  }
  const V3<T> S1 = P.s1() * z.s1, S2 = P.s2() * z.s2;
  const T r3 = r * r * r;
  if (P.terms & TERM_SO) {
    const V3<T> L = cross(z.r, z.p);
    const V3<T> Sig = P.g1() * S1 + P.g2() * S2;
    H = H + eta * dot(L, Sig) / r3;
  }
  if (P.terms & TERM_S1S2) {  // eq (3) x eta
    H = H + eta * (T(3) * dot(S1, n) * dot(S2, n) - dot(S1, S2)) / r3;
  }
  if (P.terms & TERM_QM) {  // eqs (4), (5) x eta, x kq_i
    H = H + eta * P.kq1 / (T(2) * r3 * P.beta) * (T(3) * dot(S1, n) * dot(S1, n) - dot(S1, S1));
    H = H + eta * P.kq2 * P.beta / (T(2) * r3) * (T(3) * dot(S2, n) * dot(S2, n) - dot(S2, S2));
  }
  return H;
}

// Total angular momentum J = r x p + S1 + S2.
template <class T> V3<T> total_J(const State<T>& z, const Params<T>& P) {
  return cross(z.r, z.p) + P.s1() * z.s1 + P.s2() * z.s2;
}

// ---- partial derivatives of H, term by term ---------------------------------
// Rules used: d(1/r^k)/dr = -k n / r^(k+1);  d(n.p)/dr = (p - (n.p) n)/r;
// d(S.n)/dr = (S - (S.n) n)/r;  d(a.(b x c)) cyclic.
template <class T> struct Grad { V3<T> dHdr, dHdp, dHdS1, dHdS2; };

template <class T> Grad<T> gradient(const State<T>& z, const Params<T>& P) {
  const T eta = P.eta();
  const T r = o_sqrt(dot(z.r, z.r));
  const V3<T> n = (T(1) / r) * z.r;
  const V3<T>& p = z.p;
  const T p2 = dot(p, p);
  const T np = dot(n, p);
  const V3<T> dnp = (T(1) / r) * (p - np * n);  // d(n.p)/dr
  const T r2 = r * r, r3 = r2 * r, r4 = r3 * r;
  const V3<T> zero = {T(0), T(0), T(0)};
  Grad<T> g;
  // H_N = p2/2 - 1/r
  g.dHdp = p;
  g.dHdr = (T(1) / r2) * n;
  g.dHdS1 = zero;
  g.dHdS2 = zero;
  if (P.terms & TERM_1PN) {
    // (3eta-1)/8 p2^2
    g.dHdp = g.dHdp + ((T(3) * eta - T(1)) / T(2) * p2) * p;
    // -[(3+eta) p2 + eta np^2]/(2r)
    g.dHdp = g.dHdp - (T(1) / r) * ((T(3) + eta) * p + (eta * np) * n);
    g.dHdr = g.dHdr + (((T(3) + eta) * p2 + eta * np * np) / (T(2) * r2)) * n - (eta * np / r) * dnp;
    // +1/(2 r^2)
    g.dHdr = g.dHdr - (T(1) / r3) * n;
  }
  if (P.terms & TERM_2PN) {
    const T c3 = (T(1) - T(5) * eta + T(5) * eta * eta) / T(16);
    const T d1 = T(5) - T(20) * eta - T(3) * eta * eta;
    const T e2 = eta * eta;
    // c3 p2^3
    g.dHdp = g.dHdp + (T(6) * c3 * p2 * p2) * p;
    // A/(8r), A = d1 p2^2 - 2 eta^2 np^2 p2 - 3 eta^2 np^4
    const T A = d1 * p2 * p2 - T(2) * e2 * np * np * p2 - T(3) * e2 * np * np * np * np;
    const V3<T> dAdp = (T(4) * d1 * p2) * p - (T(4) * e2 * np * p2) * n - (T(4) * e2 * np * np) * p
                       - (T(12) * e2 * np * np * np) * n;
    const T dAdnp = -T(4) * e2 * np * p2 - T(12) * e2 * np * np * np;
    g.dHdp = g.dHdp + (T(1) / (T(8) * r)) * dAdp;
    g.dHdr = g.dHdr + (dAdnp / (T(8) * r)) * dnp - (A / (T(8) * r2)) * n;
    // B/(2 r^2), B = (5+8eta) p2 + 3 eta np^2
    const T B = (T(5) + T(8) * eta) * p2 + T(3) * eta * np * np;
    g.dHdp = g.dHdp + (T(1) / (T(2) * r2)) * ((T(2) * (T(5) + T(8) * eta)) * p + (T(6) * eta * np) * n);
    g.dHdr = g.dHdr + (T(6) * eta * np / (T(2) * r2)) * dnp - (B / r3) * n;
    // -(1+3eta)/(4 r^3)
    g.dHdr = g.dHdr + (T(3) * (T(1) + T(3) * eta) / (T(4) * r4)) * n;
  }
  const V3<T> S1 = P.s1() * z.s1, S2 = P.s2() * z.s2;
  if (P.terms & TERM_SO) {
    // eta (r x p).Sig / r^3 = eta p.(Sig x r)/r^3 = eta r.(p x Sig)/r^3
    const V3<T> L = cross(z.r, p);
    const V3<T> Sig = P.g1() * S1 + P.g2() * S2;
    g.dHdp = g.dHdp + (eta / r3) * cross(Sig, z.r);
    g.dHdr = g.dHdr + (eta / r3) * cross(p, Sig) - (T(3) * eta * dot(L, Sig) / r4) * n;
    g.dHdS1 = g.dHdS1 + (eta * P.g1() / r3) * L;
    g.dHdS2 = g.dHdS2 + (eta * P.g2() / r3) * L;
  }
  if (P.terms & TERM_S1S2) {
    const T a = dot(S1, n), b = dot(S2, n);
    const V3<T> da = (T(1) / r) * (S1 - a * n), db = (T(1) / r) * (S2 - b * n);
    g.dHdr = g.dHdr + (T(3) * eta / r3) * (b * da + a * db)
                    - (T(3) * eta * (T(3) * a * b - dot(S1, S2)) / r4) * n;
    g.dHdS1 = g.dHdS1 + (eta / r3) * ((T(3) * b) * n - S2);
    g.dHdS2 = g.dHdS2 + (eta / r3) * ((T(3) * a) * n - S1);
  }
  if (P.terms & TERM_QM) {
    const T q1 = eta * P.kq1 / (T(2) * P.beta), q2 = eta * P.kq2 * P.beta / T(2);
    const T a = dot(S1, n), b = dot(S2, n);
    const V3<T> da = (T(1) / r) * (S1 - a * n), db = (T(1) / r) * (S2 - b * n);
    g.dHdr = g.dHdr + (T(6) * q1 * a / r3) * da - (T(3) * q1 * (T(3) * a * a - dot(S1, S1)) / r4) * n;
    g.dHdr = g.dHdr + (T(6) * q2 * b / r3) * db - (T(3) * q2 * (T(3) * b * b - dot(S2, S2)) / r4) * n;
    g.dHdS1 = g.dHdS1 + (q1 / r3) * ((T(6) * a) * n - T(2) * S1);
    g.dHdS2 = g.dHdS2 + (q2 / r3) * ((T(6) * b) * n - T(2) * S2);
  }
  return g;
}

// 2.5PN radiation reaction, the a_2.5PN of eq (6) ("the acceleration from the H_2.5PN radiation
// reaction in ADM coordinates").  PAPER.md does not print it (it points to Levin et al. 2011); DESIGN.md reading
// R21 takes the leading-order radiation-reaction acceleration in its general two-parameter gauge form (Iyer & Will
// 1993, 1995), per unit reduced mass and with v = p at this order,
//   a_RR = (8/5) eta / r^3 * { (n.p) n [a1 p^2 + a2 / r + a3 (n.p)^2] - p [b1 p^2 + b2 / r + b3 (n.p)^2] },
//   a1 = 3 + 3 B, a2 = 23/3 + 2 A - 3 B, a3 = -5 B, b1 = 2 + A, b2 = 2 - A, b3 = -3 - 3 A,
// in the ADM gauge of Schaefer (1985), (A, B) = (5/3, 3): a = (12, 2, -15), b = (11/3, 1/3, -8).
// Every gauge gives the same orbit-averaged energy and angular momentum fluxes (Peters & Mathews 1963, Peters 1964),
// which is what the pins check; the gauge itself is a reading.
template <class T> V3<T> rr_force(const State<T>& z, const Params<T>& P) {
  const T A = T(5) / T(3), B = T(3);
  const T a1 = T(3) + T(3) * B, a2 = T(23) / T(3) + T(2) * A - T(3) * B, a3 = T(0) - T(5) * B;
  const T b1 = T(2) + A, b2 = T(2) - A, b3 = T(0) - T(3) - T(3) * A;
  const T r = o_sqrt(dot(z.r, z.r));
  const V3<T> n = (T(1) / r) * z.r;
  const T p2 = dot(z.p, z.p);
  const T np = dot(n, z.p);
  const T ca = a1 * p2 + a2 / r + a3 * np * np;
  const T cb = b1 * p2 + b2 / r + b3 * np * np;
  return (T(8) * P.eta() / (T(5) * r * r * r)) * ((np * ca) * n - cb * z.p);
}

// Equations of motion, eqs (6)-(7):
// dr/dt = dH/dp, dp/dt = -dH/dr (+ a_2.5PN with TERM_RR), dS_i/dt = Omega_i x S_i, Omega_i = dH/dS_i.
// |S_i| is a parameter, so dS_i_hat/dt = Omega_i x S_i_hat.
// With TERM_RR also dW/dt = (dr/dt).a_2.5PN and dG/dt = r x a_2.5PN (see Diss).
template <class T> State<T> rhs(const State<T>& z, const Params<T>& P) {
  const Grad<T> g = gradient(z, P);
  const V3<T> zero = {T(0), T(0), T(0)};
  State<T> f = {g.dHdp, zero - g.dHdr, cross(g.dHdS1, z.s1), cross(g.dHdS2, z.s2), {T(0), zero}};
  if (P.terms & TERM_RR) {
    const V3<T> F = rr_force(z, P);
    f.p = f.p + F;
    f.d.w = dot(g.dHdp, F);
    f.d.g = cross(z.r, F);
  }
  return f;
}

// Classical RK4 (c = 0, 1/2, 1/2, 1; b = 1/6, 1/3, 1/3, 1/6); R9.
template <class T> State<T> rk4_step(const State<T>& z, T h, const Params<T>& P) {
  const State<T> k1 = rhs(z, P);
  const State<T> k2 = rhs(z + (h / T(2)) * k1, P);
  const State<T> k3 = rhs(z + (h / T(2)) * k2, P);
  const State<T> k4 = rhs(z + h * k3, P);
  return z + (h / T(6)) * (k1 + T(2) * k2 + T(2) * k3 + k4);
}

// Explicit Runge-Kutta step with a general Butcher tableau: k_i = f(z + h sum_j a_ij k_j), j < i;
// z' = z + h sum_i b_i k_i.  Plain loops over the tableau, every k_i stored.
struct Tableau { int stages; const double* c; const double* a; const double* b; };  // a: row-major [stages][stages]

// The paper integrates with "RK5" without giving a tableau or a step size; reading R9
// takes Butcher's classical six-stage fifth-order method (J. C. Butcher 1964; c = 0, 1/4, 1/4,
// 1/2, 3/4, 1; b = 7/90, 0, 32/90, 12/90, 32/90, 7/90).  Its 17 order conditions up to order five are
// checked on these very arrays in tests/test_oracle_integrator.py.
inline const Tableau& tableau_rk5() {
  static const double c[6] = {0.0, 1.0 / 4, 1.0 / 4, 1.0 / 2, 3.0 / 4, 1.0};
  static const double a[36] = {
      0, 0, 0, 0, 0, 0,
      1.0 / 4, 0, 0, 0, 0, 0,
      1.0 / 8, 1.0 / 8, 0, 0, 0, 0,
      0, -1.0 / 2, 1.0, 0, 0, 0,
      3.0 / 16, 0, 0, 9.0 / 16, 0, 0,
      -3.0 / 7, 2.0 / 7, 12.0 / 7, -12.0 / 7, 8.0 / 7, 0};
  static const double b[6] = {7.0 / 90, 0, 32.0 / 90, 12.0 / 90, 32.0 / 90, 7.0 / 90};
  static const Tableau T = {6, c, a, b};
  return T;
}
inline const Tableau& tableau_rk4() {
  static const double c[4] = {0.0, 0.5, 0.5, 1.0};
  static const double a[16] = {0, 0, 0, 0, 0.5, 0, 0, 0, 0, 0.5, 0, 0, 0, 0, 1.0, 0};
  static const double b[4] = {1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6};
  static const Tableau T = {4, c, a, b};
  return T;
}

template <class T> State<T> rk_step(const State<T>& z, T h, const Params<T>& P, const Tableau& tb) {
  State<T> k[8];
  for (int i = 0; i < tb.stages; ++i) {
    State<T> zi = z;
    for (int j = 0; j < i; ++j) {
      const double aij = tb.a[i * tb.stages + j];
      if (aij != 0.0) zi = zi + (h * T(aij)) * k[j];
    }
    k[i] = rhs(zi, P);
  }
  State<T> out = z;
  for (int i = 0; i < tb.stages; ++i)
    if (tb.b[i] != 0.0) out = out + (h * T(tb.b[i])) * k[i];
  return out;
}

// integrator: 0 = classical RK4 (BASELINE), 1 = Butcher's RK5 (the paper's "RK5", reading R9).
template <class T> State<T> base_step(const State<T>& z, T h, const Params<T>& P, int integrator) {
  return integrator == 1 ? rk_step(z, h, P, tableau_rk5()) : rk4_step(z, h, P);
}

// ---- manifold correction ------------------------------------------------------
template <class T> inline V3<T> unit(V3<T> s) { return (T(1) / o_sqrt(dot(s, s))) * s; }

// Reference integrals captured at the start.
template <class T> struct Refs { T E0; V3<T> J0; };
template <class T> Refs<T> references(const State<T>& z, const Params<T>& P) { return {hamiltonian(z, P), total_J(z, P)}; }

// Generic dense solve A x = b, Gaussian elimination with partial pivoting.
template <class T, int N> bool solve_dense(T A[N][N], T b[N], T x[N]) {
  for (int c = 0; c < N; ++c) {
    int piv = c;
    for (int i = c + 1; i < N; ++i)
      if (o_abs(A[i][c]) > o_abs(A[piv][c])) piv = i;
    if (!(o_abs(A[piv][c]) > T(0))) return false;
    if (piv != c) {
      for (int j = 0; j < N; ++j) { T t = A[c][j]; A[c][j] = A[piv][j]; A[piv][j] = t; }
      T t = b[c]; b[c] = b[piv]; b[piv] = t;
    }
    for (int i = c + 1; i < N; ++i) {
      const T f = A[i][c] / A[c][c];
      for (int j = c; j < N; ++j) A[i][j] = A[i][j] - f * A[c][j];
      b[i] = b[i] - f * b[c];
    }
  }
  for (int i = N - 1; i >= 0; --i) {
    T s = b[i];
    for (int j = i + 1; j < N; ++j) s = s - A[i][j] * x[j];
    x[i] = s / A[i][i];
  }
  return true;
}

// Mode 2: the paper's momentum-position dual scaling, eqs (11)-(13), read as the
// exact root H = E0, |J| = J0 (R5): p <- alpha p*, r <- beta_s r*.
// With v = 1/beta_s and gamma = alpha beta_s: |J|^2 = gamma^2 L.L + 2 gamma L.S
// + S.S is a quadratic for gamma; v follows from Newton on g(v) = H(r*/v,
// gamma v p*) - E0 started at v = 1 (R6, R7).  Returns false when the
// step is skipped (no real root / not converged / |v-1| > 1e-3).
template <class T>
bool dual_scaling(State<T>& z, const Params<T>& P, const Refs<T>& R, int newton_iters, T newton_tol) {
  const V3<T> S = P.s1() * z.s1 + P.s2() * z.s2;
  const V3<T> L = cross(z.r, z.p);
  const T LL = dot(L, L), LS = dot(L, S), SS = dot(S, S), J02 = dot(R.J0, R.J0);
  const T disc = LS * LS - LL * (SS - J02);
  if (!(disc >= T(0)) || !(LL > T(0))) return false;
  const T sgn = (LL + LS >= T(0)) ? T(1) : T(-1);
  const T gamma = (sgn * o_sqrt(disc) - LS) / LL;
  T v = T(1), dv = T(0);
  for (int it = 0; it < newton_iters; ++it) {
    State<T> zs = z;
    zs.r = (T(1) / v) * z.r;
    zs.p = (gamma * v) * z.p;
    const T g = hamiltonian(zs, P) - R.E0;
    const Grad<T> G = gradient(zs, P);
    const T dg = gamma * dot(z.p, G.dHdp) - dot(z.r, G.dHdr) / (v * v);
    dv = T(0) - g / dg;
    v = v + dv;
  }
  if (!o_finite(v) || !(o_abs(dv) <= newton_tol) || !(o_abs(v - T(1)) <= T(1) / T(1000))) return false;
  z.r = (T(1) / v) * z.r;
  z.p = (gamma * v) * z.p;
  return true;
}

// Mode 3: minimal-norm (identity metric, R14) Gauss-Newton projection
// of (r, p) onto {H = E0, r x p = J0 - S1 - S2} -- Nacozy's least-squares
// shortest-path correction applied to the four orbital integrals.
// Constraints phi = (H - E0, r x p - Lt); rows of the 4 x 6 Jacobian D are
// (dH/dr, dH/dp) and, for component k, (p x e_k, e_k x r).  Update
// (dr, dp) = -D^T (D D^T)^-1 phi.
// Iteration control as in the paper (R6): Newton
// steps are repeated until the last update is below the tolerance epsilon,
// |(dr, dp)|_2 <= newton_tol * |p|_2 (p of the point the step was computed at),
// at most newton_iters times.  The step that meets the test is still applied.
// Returns the number of steps taken.
template <class T>
int project_six(State<T>& z, const Params<T>& P, const Refs<T>& R, int newton_iters, T newton_tol) {
  const V3<T> e[3] = {{T(1), T(0), T(0)}, {T(0), T(1), T(0)}, {T(0), T(0), T(1)}};
  int done = 0;
  for (int it = 0; it < newton_iters; ++it) {
    const V3<T> Lt = R.J0 - P.s1() * z.s1 - P.s2() * z.s2;
    const Grad<T> G = gradient(z, P);
    V3<T> Dr[4], Dp[4];
    Dr[0] = G.dHdr; Dp[0] = G.dHdp;
    for (int k = 0; k < 3; ++k) { Dr[k + 1] = cross(z.p, e[k]); Dp[k + 1] = cross(e[k], z.r); }
    const V3<T> dL = cross(z.r, z.p) - Lt;
    T phi[4] = {hamiltonian(z, P) - R.E0, dL.x, dL.y, dL.z};
    T A[4][4], lam[4];
    for (int i = 0; i < 4; ++i)
      for (int j = 0; j < 4; ++j) A[i][j] = dot(Dr[i], Dr[j]) + dot(Dp[i], Dp[j]);
    if (!solve_dense<T, 4>(A, phi, lam)) return done;
    V3<T> dr = {T(0), T(0), T(0)}, dp = {T(0), T(0), T(0)};
    for (int i = 0; i < 4; ++i) { dr = dr + lam[i] * Dr[i]; dp = dp + lam[i] * Dp[i]; }
    const T step2 = dot(dr, dr) + dot(dp, dp);
    const T scale2 = dot(z.p, z.p);
    z.r = z.r - dr;
    z.p = z.p - dp;
    ++done;
    if (!(step2 > newton_tol * newton_tol * scale2)) break;  // converged (or non-finite: stop)
  }
  return done;
}

// Correction operator C_mode: 0 none; 1 eq (10);
// 2 eq (10) then dual scaling; 3 eq (10) then six-integral projection.
// Order: spins first, then (r, p) with the corrected spins.
// Returns false only when mode 2 skipped its orbital part; *gn_steps (optional)
// receives the number of Gauss-Newton steps mode 3 took.
template <class T>
bool correct(State<T>& z, const Params<T>& P, const Refs<T>& R, int mode, int newton_iters, T newton_tol,
             int* gn_steps = nullptr) {
  if (gn_steps) *gn_steps = 0;
  if (mode >= 1) { z.s1 = unit(z.s1); z.s2 = unit(z.s2); }  // eq (10)
  if (mode == 2) return dual_scaling(z, P, R, newton_iters, newton_tol);
  if (mode == 3) {
    const int k = project_six(z, P, R, newton_iters, newton_tol);
    if (gn_steps) *gn_steps = k;
  }
  return true;
}

// ---- whole-orbit driver ---------------------
enum : int32_t { ST_OK = 0, ST_MERGED = 1, ST_UNBOUND = 2, ST_NONFINITE = 3, ST_NEWTON_FLAG = 256 };

template <class T> inline bool finite_state(const State<T>& z) {
  const T v[12] = {z.r.x, z.r.y, z.r.z, z.p.x, z.p.y, z.p.z, z.s1.x, z.s1.y, z.s1.z, z.s2.x, z.s2.y, z.s2.z};
  for (int i = 0; i < 12; ++i)
    if (!o_finite(v[i])) return false;
  return true;
}

struct Options {
  int mode;             // correction mode 0..3
  int renorm_interval;  // steps between shadow renormalisations (BASELINE config 1: 100)
  int newton_iters;     // Newton iteration cap (mode 3) / fixed count (mode 2), R6
  double newton_tol;    // epsilon of PAPER.md:197: mode 3 termination test, mode 2 convergence flag
  double r_merge, r_escape;  // DESIGN.md R13
  int integrator;       // 0 classical RK4, 1 Butcher RK5 (R9)
};

template <class T> struct OrbitResult {
  State<T> z;            // final (or frozen) main state
  T inv0[6], inv1[6];    // E, Jx, Jy, Jz, |S1hat|, |S2hat| at start / end
  T fli;                 // log10 d(t)/d(0), accumulated over renormalisations
  int32_t status;
  int64_t steps_done;
  int64_t gn_steps;      // Gauss-Newton steps of mode 3 over all accepted steps, orbit + shadow
  State<T> zs;           // final shadow state (= z without a shadow) and the integrals it is corrected onto;
  T Es0; V3<T> Js0;      //   reported so that the shadow's own invariants can be pinned (tests only)
};

template <class T> inline void six_integrals(const State<T>& z, const Params<T>& P, T out[6]) {
  const V3<T> J = total_J(z, P);
  out[0] = hamiltonian(z, P); out[1] = J.x; out[2] = J.y; out[3] = J.z;
  out[4] = o_sqrt(dot(z.s1, z.s1)); out[5] = o_sqrt(dot(z.s2, z.s2));
}

// sampler(s, z): optional callback, called after every sample_interval-th step index (k = interval, 2 interval,
// ...) with the orbit's current state -- the frozen state once the orbit has been dropped.
template <class T, class Sampler>
OrbitResult<T> integrate_orbit(State<T> z, const Params<T>& P, T h, int64_t n_steps, T shadow_eps, const Options& O,
                               int64_t sample_interval, Sampler sampler) {
  OrbitResult<T> out;
  const bool shadow = !(shadow_eps == T(0));
  const bool rr = (P.terms & TERM_RR) != 0;
  const V3<T> zero3 = {T(0), T(0), T(0)};
  z.d = {T(0), zero3};
  // With radiation reaction the manifold moves: the correction targets E0 + W, J0 + G (integral invariant relation,
  // PAPER.md:221), W and G being the dissipation integrals the step itself has just advanced.
  auto moved = [&](const Refs<T>& R0, const State<T>& zz) { return rr ? Refs<T>{R0.E0 + zz.d.w, R0.J0 + zz.d.g} : R0; };
  if (O.mode >= 1) { z.s1 = unit(z.s1); z.s2 = unit(z.s2); }
  Refs<T> R = references(z, P);
  six_integrals(z, P, out.inv0);
  State<T> zs = z;
  Refs<T> Rs = R;
  T d0 = T(0), acc = T(0);
  if (shadow) {
    zs.r.x = zs.r.x + shadow_eps;
    d0 = o_abs(shadow_eps);
    Rs = references(zs, P);
  }
  int32_t status = ST_OK, flag = 0;
  int64_t k = 0, gn_total = 0;
  while (k < n_steps) {
    int gn = 0, gns = 0;
    State<T> zn = base_step(z, h, P, O.integrator);
    if (!correct(zn, P, moved(R, zn), O.mode, O.newton_iters, T(O.newton_tol), &gn)) flag = ST_NEWTON_FLAG;
    State<T> zsn = zs;
    if (shadow) {
      zsn = base_step(zs, h, P, O.integrator);
      correct(zsn, P, moved(Rs, zsn), O.mode, O.newton_iters, T(O.newton_tol), &gns);
    }
    // status check on the completed step (R13); on failure keep the last good state
    if (!finite_state(zn) || !finite_state(zsn)) { status = ST_NONFINITE; break; }
    const T rr = o_sqrt(dot(zn.r, zn.r));
    if (rr < T(O.r_merge)) { status = ST_MERGED; break; }
    if (rr > T(O.r_escape)) { status = ST_UNBOUND; break; }
    z = zn; zs = zsn; ++k; gn_total += gn + gns;
    if (sample_interval > 0 && k % sample_interval == 0) sampler(k / sample_interval - 1, z);
    if (shadow && O.renorm_interval > 0 && (k % O.renorm_interval) == 0) {
      const State<T> dz = zs - z;
      const T d = o_sqrt(norm12sq(dz));
      if (!(d > T(0)) || !o_finite(d)) { status = ST_NONFINITE; break; }
      acc = acc + o_log10(d / d0);
      zs = z + (d0 / d) * dz;
      if (O.mode >= 1) { zs.s1 = unit(zs.s1); zs.s2 = unit(zs.s2); }
      Rs = references(zs, P);  // DESIGN.md R11
      zs.d = {T(0), zero3};    // its dissipation integrals restart with its references
    }
  }
  if (sample_interval > 0)   // a dropped orbit keeps reporting its frozen state
    for (int64_t kk = (k / sample_interval + 1) * sample_interval; kk <= n_steps; kk += sample_interval)
      sampler(kk / sample_interval - 1, z);
  out.z = z;
  six_integrals(z, P, out.inv1);
  out.fli = shadow ? acc + o_log10(o_sqrt(norm12sq(zs - z)) / d0) : T(0);
  out.status = status | flag;
  out.steps_done = k;
  out.gn_steps = gn_total;
  out.zs = zs; out.Es0 = Rs.E0; out.Js0 = Rs.J0;
  return out;
}

template <class T>
OrbitResult<T> integrate_orbit(State<T> z, const Params<T>& P, T h, int64_t n_steps, T shadow_eps, const Options& O) {
  return integrate_orbit<T>(z, P, h, n_steps, shadow_eps, O, 0, [](int64_t, const State<T>&) {});
}

}  // namespace pn_oracle
