/* A plain C99 client of liblpc.so: include/lpc.h compiled by a C compiler, and the five calls the north star names
 * (lpc_create_lattice / lpc_set_site_params / lpc_step_n / lpc_read_fid / lpc_moments) run from C with nothing but the
 * CUDA runtime for the workspace allocation.
 *
 * The lattice is homogeneous with a uniform chemical shift, for which the paper fixes the answers in closed form:
 *   G[n] = exp(i omega n dt)                (Eq. 8 / Eq. 12: every spin precesses at the same rate)
 *   D_d  = alpha a^2 / (6 dt)               (Eq. 7, with d = 3)
 * so the program checks itself and prints "OK".  Exit code 0 = pass, 1 = a wrong number, 2 = an error code from the ABI.
 *
 * Build (tests/test_c_client.py):  gcc -std=c99 -Wall -Wextra -Werror -pedantic -Iinclude -isystem $CUDA/include lpc_client.c
 *                                  -Lpaper_2603_22553_b200 -llpc -L$CUDA/lib64 -lcudart -lm
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "lpc.h"

#define CHECK(call)                                                                  \
  do {                                                                               \
    int rc_ = (call);                                                                \
    if (rc_ != LPC_OK) {                                                             \
      fprintf(stderr, "%s -> %d: %s\n", #call, rc_, lpc_last_error());               \
      return 2;                                                                      \
    }                                                                                \
  } while (0)

int main(void) {
  const int nx = 24, ny = 16, nz = 40, steps = 21;
  const double dt = 5e-6, alpha = 0.75, omega = -9000.0;
  const size_t n = (size_t)nx * ny * nz;
  lpc_config cfg;
  size_t bytes = 0, i;
  void* ws = NULL;
  lpc_lattice* lat = NULL;
  double *dF, *om, *fid, *vacf, D[3], worst = 0.0;
  uint8_t* blocked;
  int k, d;

  memset(&cfg, 0, sizeof(cfg));
  cfg.nx = nx; cfg.ny = ny; cfg.nz = nz;
  cfg.n_moments = 3;
  cfg.dt = dt; cfg.a = 1.0; cfg.alpha = alpha;
  cfg.max_steps = steps;
  cfg.stream = NULL;

  /* argument checking needs no GPU */
  if (lpc_workspace_bytes(NULL, &bytes) != LPC_EINVAL || lpc_last_error()[0] == '\0') return 1;
  CHECK(lpc_workspace_bytes(&cfg, &bytes));
  if (cudaMalloc(&ws, bytes) != cudaSuccess) {
    fprintf(stderr, "cudaMalloc of %zu bytes failed\n", bytes);
    return 2;
  }
  CHECK(lpc_create_lattice(&cfg, ws, bytes, &lat));

  dF = (double*)calloc(n, sizeof(double));
  om = (double*)malloc(n * sizeof(double));
  blocked = (uint8_t*)calloc(n, 1);
  fid = (double*)malloc(2 * (size_t)(steps + 1) * sizeof(double));
  vacf = (double*)malloc(3 * (size_t)(steps + 1) * sizeof(double));
  if (!dF || !om || !blocked || !fid || !vacf) return 2;
  for (i = 0; i < n; ++i) om[i] = omega;

  CHECK(lpc_set_site_params(lat, dF, blocked, om, NULL));
  CHECK(lpc_step_n(lat, steps));
  if (lpc_steps_done(lat) != steps) return 1;
  CHECK(lpc_read_fid(lat, 0, steps + 1, fid));
  CHECK(lpc_moments(lat, steps + 1, vacf, D));

  for (k = 0; k <= steps; ++k) {
    const double er = fid[2 * k] - cos(omega * dt * k), ei = fid[2 * k + 1] - sin(omega * dt * k);
    const double e = sqrt(er * er + ei * ei);
    if (e > worst) worst = e;
  }
  printf("max |G[n] - exp(i omega n dt)| = %.3e\n", worst);
  if (worst > 1e-12) return 1;
  for (d = 0; d < 3; ++d) {
    const double want = alpha / (6.0 * dt);
    printf("D[%d] = %.12g (Eq. 7: %.12g)\n", d, D[d], want);
    if (fabs(D[d] - want) > 1e-9 * want) return 1;
    if (fabs(vacf[d * (steps + 1)] - alpha / 3.0) > 1e-12) return 1; /* Z_d[1] = alpha a^2 / 3 */
  }
  /* errors come back as codes, never as a crash */
  if (lpc_step_n(lat, 1) != LPC_EINVAL) return 1; /* over max_steps */
  if (lpc_read_fid(lat, 0, steps + 5, fid) != LPC_EINVAL) return 1;

  lpc_destroy(lat);
  cudaFree(ws);
  free(dF); free(om); free(blocked); free(fid); free(vacf);
  printf("OK\n");
  return 0;
}
