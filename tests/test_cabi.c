/* test_cabi.c — a plain C program against include/hard.h (no Python, no torch): the five calls that
 * BASELINE.json's north_star names, on the Sod shock tube of PAPER.md P:200-203 eq.20 with 64 cells.
 * Compiled by tests/test_boundary_cpu.py (gcc -I include, linked against libhard_b200.so) on the CPU box and
 * run on the GPU box by tests/test_gpu_api.py.  Exit code 0 = all checks passed.
 *
 * Hand values (written from the definitions, not from any implementation):
 *   cell size dx = 1/64; left state (rho, u, p) = (1, 0, 1), right (0.125, 0, 0.1), gamma = 1.4;
 *   c_s = sqrt(gamma p / rho): left sqrt(1.4) = 1.18321595661992..., right sqrt(1.12) = 1.0583...;
 *   lambda = max (|u| + c_s)/dx = 64 sqrt(1.4)  =>  hard_max_dt = 1/lambda = 0.01320529...  (G6).
 *   After a few steps no wave has reached the ends (outflow, G10), so total mass and energy are what they were.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "hard.h"

#define N 64
#define CHECK(cond, msg)                                                        \
  do {                                                                          \
    if (!(cond)) { fprintf(stderr, "FAIL: %s (%s)\n", msg, h ? hard_last_error(h) : hard_last_error(NULL)); return 1; } \
  } while (0)

int main(void) {
  const double gamma = 1.4;
  double rho[N], mx[N], my[N], mz[N], E[N], out[5][N];
  double mass0 = 0.0, en0 = 0.0, mass1 = 0.0, en1 = 0.0, dt = 0.0, t = 0.0;
  long long steps = 0;
  int i, rc;
  hard_ctx* h = hard_create(N, 1, 1, gamma, HARD_BC_OUTFLOW);
  CHECK(h != NULL, "hard_create");
  for (i = 0; i < N; ++i) {
    const int left = (i + 0.5) / N < 0.5;
    rho[i] = left ? 1.0 : 0.125;
    mx[i] = my[i] = mz[i] = 0.0;
    E[i] = (left ? 1.0 : 0.1) / (gamma - 1.0);
    mass0 += rho[i];
    en0 += E[i];
  }
  rc = hard_set_state(h, rho, mx, my, mz, E);             /* host pointers */
  CHECK(rc == HARD_OK, "hard_set_state");
  rc = hard_max_dt(h, &dt);
  CHECK(rc == HARD_OK, "hard_max_dt");
  CHECK(fabs(dt - 1.0 / (64.0 * sqrt(1.4))) <= 1e-14 * dt, "hard_max_dt = dx / sqrt(gamma p_L / rho_L)");
  rc = hard_step(h, 0.4, 5);
  CHECK(rc == HARD_OK, "hard_step");
  rc = hard_get_state(h, out[0], out[1], out[2], out[3], out[4]);
  CHECK(rc == HARD_OK, "hard_get_state");
  rc = hard_get_time(h, &t, &steps);
  CHECK(rc == HARD_OK && steps == 5 && t > 4.0 * 0.4 * dt * 0.5 && t < 5.0 * 0.4 * dt * 1.0001, "hard_get_time");
  for (i = 0; i < N; ++i) { mass1 += out[0][i]; en1 += out[4][i]; }
  CHECK(fabs(mass1 - mass0) <= 1e-13 * mass0, "mass conserved while no wave has reached the ends");
  CHECK(fabs(en1 - en0) <= 1e-13 * en0, "energy conserved while no wave has reached the ends");
  CHECK(out[0][0] == 1.0 && out[0][N - 1] == 0.125, "the far field is untouched");
  CHECK(out[1][N / 2] > 0.0 && out[0][N / 2 - 1] < 1.0 && out[0][N / 2] > 0.125, "the diaphragm has burst: flow to the right");
  for (i = 0; i < N; ++i) CHECK(out[2][i] == 0.0 && out[3][i] == 0.0, "transverse momenta stay zero in 1-D (G11, G15)");
  rc = hard_max_dt(h, &dt);
  CHECK(rc == HARD_OK && dt > 0.0 && dt < 1.0 / (64.0 * sqrt(1.4)), "the shock raises the max wave speed");
  CHECK(hard_step(h, -1.0, 1) == HARD_ERR_ARG, "hard_step rejects cfl <= 0");
  CHECK(hard_destroy(h) == HARD_OK, "hard_destroy");
  h = NULL;
  printf("test_cabi ok: dt0 = %.17g, t = %.17g after %lld steps, mass %.17g\n", 1.0 / (64.0 * sqrt(1.4)), t, steps, mass1);
  return 0;
}
