/* Driver for an AddressSanitizer + UndefinedBehaviorSanitizer build of the CPU oracle: it is compiled
 * TOGETHER with oracle/lpc_oracle.c (tests/test_oracle_pins.py::test_oracle_is_clean_under_asan_and_ubsan) and walks every
 * entry point on small lattices with ragged shapes, degenerate axes, walls, link factors and moment fields.  Any
 * out-of-bounds access, use after free, signed overflow or misaligned access aborts the run; leaks fail it at exit. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct {
  int32_t nx, ny, nz;
  int32_t bc[3];
  double dt, a, alpha;
} lpco_config;
typedef struct lpco_state lpco_state;

lpco_state* lpco_create_links(const lpco_config*, const double*, const uint8_t*, const double*, const double*, int, int64_t);
lpco_state* lpco_create(const lpco_config*, const double*, const uint8_t*, const double*, int, int64_t);
void lpco_destroy(lpco_state*);
int lpco_step(lpco_state*, int64_t);
int lpco_set_g(lpco_state*, const double*);
int lpco_propagate_real(const lpco_state*, const double*, double*, int64_t);
int64_t lpco_equilibrate(const lpco_state*, double*, double, int64_t, double*);
int64_t lpco_steps(const lpco_state*);
double lpco_partition_sum(const lpco_state*);
void lpco_get_pi(const lpco_state*, double*);
void lpco_get_stay(const lpco_state*, double*);
void lpco_get_p_in(const lpco_state*, int, double*);
void lpco_get_g(const lpco_state*, double*);
int lpco_get_P(const lpco_state*, int, double*);
int lpco_get_u(const lpco_state*, int, double*);
int lpco_get_fid(const lpco_state*, int64_t, int64_t, double*, double*);
int lpco_get_moments(const lpco_state*, int64_t, double*, double*);
int64_t lpco_neighbor(const lpco_config*, int64_t, int, int);

static double urand(uint64_t* s) { /* splitmix64 */
  uint64_t z = (*s += 0x9e3779b97f4a7c15ull);
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  z ^= z >> 31;
  return (double)(z >> 11) / 9007199254740992.0;
}

static int run(int nx, int ny, int nz, int b0, int b1, int b2, int use_links, int nm, uint64_t seed) {
  const int64_t n = (int64_t)nx * ny * nz, steps = 7;
  lpco_config c = {nx, ny, nz, {b0, b1, b2}, 2e-5, 1.0, 0.8};
  double* dF = malloc(n * sizeof(double));
  double* om = malloc(n * sizeof(double));
  double* link = malloc(3 * n * sizeof(double));
  double* buf = malloc(2 * n * sizeof(double));
  double* out = malloc(2 * n * sizeof(double));
  double* fid = malloc(2 * (steps + 1) * sizeof(double));
  double* sabs = malloc((steps + 1) * sizeof(double));
  double* vacf = malloc(3 * (steps + 1) * sizeof(double));
  double* dl = malloc(16 * sizeof(double));
  uint8_t* blk = malloc(n);
  double D[3], mass = 0.0, mass2 = 0.0;
  int64_t i;
  int k, bad = 0;
  for (i = 0; i < n; ++i) {
    dF[i] = -3.0 * urand(&seed);
    om[i] = -2.5e4 * urand(&seed);
    blk[i] = (n > 4 && urand(&seed) < 0.25) ? 1 : 0;
  }
  blk[0] = 0;
  for (i = 0; i < 3 * n; ++i) link[i] = urand(&seed);
  lpco_state* st = use_links ? lpco_create_links(&c, dF, blk, om, link, nm, steps) : lpco_create(&c, dF, blk, om, nm, steps);
  if (!st) return 1;
  for (i = 0; i < n; ++i) {
    for (k = 0; k < 6; ++k) (void)lpco_neighbor(&c, i, k / 2, (k & 1) ? 1 : -1);
  }
  bad |= lpco_step(st, 3);
  for (i = 0; i < 2 * n; ++i) buf[i] = urand(&seed) - 0.5;
  bad |= lpco_set_g(st, buf);
  bad |= lpco_step(st, steps);
  bad |= (lpco_step(st, 1) == 0);                        /* over capacity must be refused */
  bad |= (lpco_steps(st) != steps);
  bad |= lpco_get_fid(st, 0, steps + 1, fid, sabs);
  bad |= (lpco_get_fid(st, 1, steps + 1, fid, sabs) == 0); /* out of range must be refused */
  lpco_get_pi(st, out); lpco_get_stay(st, out); lpco_get_g(st, out);
  for (k = 0; k < 6; ++k) lpco_get_p_in(st, k, out);
  if (nm == 3) {
    for (k = 0; k < 3; ++k) { bad |= lpco_get_P(st, k, out); bad |= lpco_get_u(st, k, out); }
    bad |= lpco_get_moments(st, steps + 1, vacf, D);
  } else {
    bad |= (lpco_get_P(st, 0, out) == 0);
  }
  for (i = 0; i < n; ++i) { buf[i] = blk[i] ? 0.0 : urand(&seed); mass += buf[i]; }
  bad |= lpco_propagate_real(st, buf, out, 5);
  for (i = 0; i < n; ++i) mass2 += out[i];
  bad |= !(fabs(mass2 - mass) <= 1e-12 * (mass + 1.0));  /* conservation */
  bad |= (lpco_equilibrate(st, buf, 0.0, 9, dl) != 9);
  bad |= !(lpco_partition_sum(st) > 0.0);
  lpco_destroy(st);
  free(dF); free(om); free(link); free(buf); free(out); free(fid); free(sabs); free(vacf); free(dl); free(blk);
  return bad;
}

int main(void) {
  int bad = 0;
  bad |= run(5, 3, 7, 0, 0, 0, 0, 3, 1);
  bad |= run(6, 4, 9, 1, 0, 1, 1, 3, 2);
  bad |= run(2, 1, 3, 0, 0, 0, 0, 3, 3);   /* degenerate axes */
  bad |= run(1, 1, 1, 0, 0, 0, 1, 0, 4);   /* a single site */
  bad |= run(4, 4, 4, 1, 1, 1, 1, 0, 5);   /* a closed box */
  bad |= (lpco_create(NULL, NULL, NULL, NULL, 0, 0) != NULL);
  printf(bad ? "FAILED\n" : "CLEAN\n");
  return bad ? 1 : 0;
}
