// mc_consts.h -- derived constants of one binary, as the kernels consume them.
//
// The kernels work with unit spins sigma_i, raw dot products and u = 1/|r|; every eta-, beta-,
// chi- and kappa-dependent factor of the Hamiltonian is folded into the
// constants below once per orbit.  Disabled terms (mc_terms bit-mask) become zero coefficients.
#pragma once
#include <stdint.h>

#ifdef __CUDACC__
#define MC_HD __host__ __device__ __forceinline__
#else
#define MC_HD inline
#endif

// Orbital part:  H_orb = P/2 - u + a1 P^2 + c3 P^3 + u [(b1 + d1 P + d2 Q) P + (b2 + d3 Q) Q]
//                        + u^2 (h1 + e1 P + e2 Q) + f1 u^3,   P = p.p, Q = (n.p)^2, u = 1/r
// Spin part (sigma_i unit spins, L = r x p, a_i = sigma_i . r, d_ij = sigma_i . sigma_j):
//   H_SO  = u^3 L.(k1 sigma1 + k2 sigma2)
//   H_12  = c12 (3 a1 a2 u^5 - d12 u^3)
//   H_ii  = q_i (3 a_i^2 u^5 - d_ii u^3)
//   Omega1 = o1 u^3 L + 3 u^5 (m12 a2 + m11 a1) r - m12 u^3 sigma2     (= dH/dS1, S1 = s1 sigma1)
//   Omega2 = o2 u^3 L + 3 u^5 (m21 a1 + m22 a2) r - m21 u^3 sigma1
//   J = L + s1 sigma1 + s2 sigma2
// Radiation reaction (2.5PN, eq (6) of the paper; R21), force per unit mu with v = p at this order:
//   F = u^3 [ (ra1 P + ra2 u + ra3 Q) (r.p) u^2 r - (rb1 P + rb2 u + rb3 Q) p ],  ra_i = (8/5) eta a_i, rb_i = (8/5) eta b_i,
//   a = (3 + 3B, 23/3 + 2A - 3B, -5B), b = (2 + A, 2 - A, -3 - 3A) with the ADM gauge (A, B) = (5/3, 3)
enum { MC_NCONST = 45 };
enum McConstIndex {
  K_A1 = 0, K_B1, K_B2, K_H1, K_C3, K_D1, K_D2, K_D3, K_E1, K_E2, K_F1,  // orbital
  K_K1, K_K2, K_C12, K_Q1, K_Q2,                                         // spin couplings in H
  K_O1, K_O2, K_M12, K_M21, K_M11, K_M22,                                // precession
  K_S1, K_S2,                                                            // spin magnitudes
  // fixed multiples of the above, so that no constant x constant product is left in the step loop
  K_2A1, K_3C3, K_2H1, K_3F1, K_2B2, K_2D2, K_4D3, K_2E2, K_2E1,         // 2 H_P, 2 H_Q, H_u polynomials
  K_3C12, K_M5C12, K_3M12, K_3M21, K_3M11, K_3M22,                        // spin-spin gradient / precession
  K_RA1, K_RA2, K_RA3, K_RB1, K_RB2, K_RB3                                 // 2.5PN radiation reaction (MC_TERM_RR)
};

struct McConsts { double v[MC_NCONST]; };

MC_HD void mc_derive_consts(double beta, double chi1, double chi2, double kq1, double kq2, uint32_t terms,
                            double* c /* [MC_NCONST] */, int stride = 1) {
  const double eta = beta / ((1.0 + beta) * (1.0 + beta));
  const double pn1 = (terms & 1u) ? 1.0 : 0.0, pn2 = (terms & 2u) ? 1.0 : 0.0;
  const double so = (terms & 4u) ? 1.0 : 0.0, ss = (terms & 8u) ? 1.0 : 0.0, qm = (terms & 16u) ? 1.0 : 0.0;
  const double s1 = chi1 * beta, s2 = chi2 / beta;          // |S_i| in units of mu M
  const double g1 = 2.0 + 1.5 / beta, g2 = 2.0 + 1.5 * beta;  // eqs (8), (9)
  c[K_A1 * stride] = pn1 * (3.0 * eta - 1.0) / 8.0;
  c[K_B1 * stride] = -pn1 * (3.0 + eta) / 2.0;
  c[K_B2 * stride] = -pn1 * eta / 2.0;
  c[K_H1 * stride] = pn1 * 0.5;
  c[K_C3 * stride] = pn2 * (1.0 - 5.0 * eta + 5.0 * eta * eta) / 16.0;
  c[K_D1 * stride] = pn2 * (5.0 - 20.0 * eta - 3.0 * eta * eta) / 8.0;
  c[K_D2 * stride] = -pn2 * eta * eta / 4.0;
  c[K_D3 * stride] = -pn2 * 3.0 * eta * eta / 8.0;
  c[K_E1 * stride] = pn2 * (5.0 + 8.0 * eta) / 2.0;
  c[K_E2 * stride] = pn2 * 1.5 * eta;
  c[K_F1 * stride] = -pn2 * (1.0 + 3.0 * eta) / 4.0;
  c[K_K1 * stride] = so * eta * g1 * s1;
  c[K_K2 * stride] = so * eta * g2 * s2;
  c[K_C12 * stride] = ss * eta * s1 * s2;
  c[K_Q1 * stride] = qm * eta * kq1 * s1 * s1 / (2.0 * beta);
  c[K_Q2 * stride] = qm * eta * kq2 * beta * s2 * s2 / 2.0;
  c[K_O1 * stride] = so * eta * g1;
  c[K_O2 * stride] = so * eta * g2;
  c[K_M12 * stride] = ss * eta * s2;
  c[K_M21 * stride] = ss * eta * s1;
  c[K_M11 * stride] = qm * eta * kq1 * s1 / beta;
  c[K_M22 * stride] = qm * eta * kq2 * beta * s2;
  c[K_S1 * stride] = s1;
  c[K_S2 * stride] = s2;
  c[K_2A1 * stride] = 2.0 * c[K_A1 * stride];
  c[K_3C3 * stride] = 3.0 * c[K_C3 * stride];
  c[K_2H1 * stride] = 2.0 * c[K_H1 * stride];
  c[K_3F1 * stride] = 3.0 * c[K_F1 * stride];
  c[K_2B2 * stride] = 2.0 * c[K_B2 * stride];
  c[K_2D2 * stride] = 2.0 * c[K_D2 * stride];
  c[K_4D3 * stride] = 4.0 * c[K_D3 * stride];
  c[K_2E2 * stride] = 2.0 * c[K_E2 * stride];
  c[K_2E1 * stride] = 2.0 * c[K_E1 * stride];
  c[K_3C12 * stride] = 3.0 * c[K_C12 * stride];
  c[K_M5C12 * stride] = -5.0 * c[K_C12 * stride];
  c[K_3M12 * stride] = 3.0 * c[K_M12 * stride];
  c[K_3M21 * stride] = 3.0 * c[K_M21 * stride];
  c[K_3M11 * stride] = 3.0 * c[K_M11 * stride];
  c[K_3M22 * stride] = 3.0 * c[K_M22 * stride];
  const double rr = (terms & 32u) ? 1.6 * eta : 0.0, gA = 5.0 / 3.0, gB = 3.0;   // Schaefer's ADM gauge
  c[K_RA1 * stride] = rr * (3.0 + 3.0 * gB);
  c[K_RA2 * stride] = rr * (23.0 / 3.0 + 2.0 * gA - 3.0 * gB);
  c[K_RA3 * stride] = rr * (-5.0 * gB);
  c[K_RB1 * stride] = rr * (2.0 + gA);
  c[K_RB2 * stride] = rr * (2.0 - gA);
  c[K_RB3 * stride] = rr * (-3.0 - 3.0 * gA);
}
