/* A plain C99 program that drives the boundary of include/mc.h without Python, torch or CUDA headers (the host-buffer
 * entry point).  Built and run by tests/test_parity_gpu.py::test_plain_c_program_drives_the_library.
 * Workload: 40 orbits shaped like BASELINE config 0 (r0 = (a,0,0), p0 = (0, f/sqrt(a), 0), tilted unit spins) with a
 * shadow, 2000 RK4 steps of h = 1, six-integral correction.  Checks what holds without an oracle: return codes, status 0,
 * all steps done, relative drift of the energy and of J below 1e-12 (north_star), unit spins, 0 < FLI < 5.8 (regular
 * orbits), and that a second identical call reproduces the first bit for bit. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "mc.h"

#define N 40

static int fail(const char* what, int rc) {
  fprintf(stderr, "c_abi_caller: %s failed: %d (%s)\n", what, rc, mc_strerror(rc));
  return 1;
}

int main(void) {
  mc_params P;
  mc_handle* h = NULL;
  int rc = mc_params_default(&P);
  if (rc) return fail("mc_params_default", rc);
  P.beta = 0.8; P.chi1 = 0.9; P.chi2 = 0.7;
  rc = mc_create(&P, &h);
  if (rc) return fail("mc_create", rc);

  static double z[12 * N], out[12 * N], out2[12 * N], inv[12 * N], fli[N], fli2[N];
  static int32_t status[N];
  static int64_t steps[N];
  for (int o = 0; o < N; ++o) {
    const double a = 15.0 + 15.0 * o / (N - 1), f = 0.85 + 0.14 * ((o * 7) % N) / (double)N;
    const double t1 = 0.3 + 0.05 * o, t2 = 2.0 - 0.03 * o;
    const double v[12] = {a, 0, 0, 0, f / sqrt(a), 0, sin(t1), 0, cos(t1), sin(t2) * 0.6, sin(t2) * 0.8, cos(t2)};
    for (int i = 0; i < 12; ++i) z[i * N + o] = v[i];
  }
  rc = mc_integrate_host(h, z, N, 1.0, 2000, MC_CORR_SIXINT, 1e-8, out, inv, fli, status, steps);
  if (rc) return fail("mc_integrate_host", rc);
  rc = mc_integrate_host(h, z, N, 1.0, 2000, MC_CORR_SIXINT, 1e-8, out2, NULL, fli2, NULL, NULL);
  if (rc) return fail("mc_integrate_host (second call)", rc);
  if (memcmp(out, out2, sizeof(out)) != 0 || memcmp(fli, fli2, sizeof(fli)) != 0) { fprintf(stderr, "not reproducible\n"); return 1; }

  double worst_e = 0, worst_j = 0, worst_s = 0;
  for (int o = 0; o < N; ++o) {
    if (status[o] != 0 || steps[o] != 2000) { fprintf(stderr, "orbit %d: status %d after %lld steps\n", o, (int)status[o], (long long)steps[o]); return 1; }
    const double e0 = inv[0 * N + o], e1 = inv[6 * N + o];
    double j0 = 0, dj = 0;
    for (int k = 1; k <= 3; ++k) { const double a = inv[k * N + o], b = inv[(6 + k) * N + o]; j0 += a * a; dj += (b - a) * (b - a); }
    worst_e = fmax(worst_e, fabs(e1 / e0 - 1.0));
    worst_j = fmax(worst_j, sqrt(dj / j0));
    worst_s = fmax(worst_s, fmax(fabs(inv[10 * N + o] - 1.0), fabs(inv[11 * N + o] - 1.0)));
    if (!(fli[o] > 0.0 && fli[o] < 5.8)) { fprintf(stderr, "orbit %d: FLI %g\n", o, fli[o]); return 1; }
  }
  mc_launch_info info;
  rc = mc_last_launch_info(h, &info);
  if (rc) return fail("mc_last_launch_info", rc);
  rc = mc_destroy(h);
  if (rc) return fail("mc_destroy", rc);
  printf("c_abi_caller ok: %d orbits x 2000 steps, |dE/E| %.2e, |dJ|/|J| %.2e, ||S|-1| %.2e, regs %d, spill bytes %d\n",
         N, worst_e, worst_j, worst_s, (int)info.regs_per_thread, (int)info.local_bytes);
  return (worst_e < 1e-12 && worst_j < 1e-12 && worst_s < 1e-14 && info.local_bytes == 0) ? 0 : 1;
}
