/*
 * lpc_oracle.c -- CPU ORACLE for the LPC3D lattice update.  TEST INFRASTRUCTURE.
 *
 * A plain, slow, double-precision restatement of what the hot path computes,
 * written from /root/reference/PAPER.md (arxiv 2603.22553) and the readings in
 * DESIGN.md.  It exists so that the CUDA library can be checked against
 * something that is not itself.  It shares NO code with
 * paper_2603_22553_b200/ (no headers, helpers, tables or packing), and only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.  It is never tuned for speed.
 *
 * Build:  gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (see oracle/build.py)
 *         -ffp-contract=off keeps every a*b+c as two roundings, so the result
 *         does not depend on whether the host has FMA.
 *
 * Notation (PAPER.md "Description of the model"):
 *   site index  i = (x*ny + y)*nz + z          (z fastest, numpy C order)
 *   dF_i        site free energy in kT  (E_i / k_B T)
 *   blocked_i   1 = carbon / inaccessible site
 *   omega_i     2 pi nu_i, rad/s               (Eq. 11 :132)
 *   alpha       global jump factor, Eq. 7
 *
 * Steps:
 *   O1  Boltzmann density pi_i                      Eq. 2
 *   O2  neighbour with boundary conditions
 *   O3  hop probability p(i->j)                     Eq. 1   PAPER.md:61, z=6 :55, alpha :101, obstacles :95
 *   O4  stay probability
 *   O5  g'_i = e^{i omega_i dt} [stay_i g_i + sum_j p(j->i) g_j]   Eq. 13
 *   O6  G[n] = sum_i g_i(n)                         Eq. 12
 *   O7  first-step moments P^d(1), u^d, Z_d[1]      Eq. 4, 5 PAPER.md:79,92; :84-86
 *   O8  Z_d[k+1] = sum_i P^d_i u^d_i ; P^d <- W P^d ; D_d   Eq. 4
 *   O9  equilibration loop rho <- W rho until max_i |rho(t+1)-rho(t)| < threshold
 *   O10 per-link mobility factor alpha_ij: p(i->j) and p(j->i) are both multiplied by the factor of
 *       the link (detailed balance kept)
 *
 * Every global sum is Neumaier-compensated, taken plane by plane (x) and the
 * plane partials combined in x order, so results do not depend on the OpenMP
 * thread count.
 *
 * Pins (tests/test_oracle_pins.py): conservation, detailed balance,
 * stationarity of Eq. 2, relaxation per connected cluster, free-diffusion
 * closed form (Eq. 7), uniform-shift single line, trajectory-enumeration brute
 * force of Eq. 8/11 and of <dx_1 dx_n> on 4^3 and smaller, Lorentz-gas first
 * lag, bounded-system sum rule, axis-permutation and translation symmetry;
 * lpco_set_g and the sum_i |g_i| tolerance-scale series against the dense
 * (Phi W)^n on <= 4^3 (P18, P19).
 * Parity unpinned: the paper's application numbers (Table 1, peak ppm), whose
 * inputs are not available.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
  int32_t nx, ny, nz;
  int32_t bc[3]; /* per axis: 0 periodic, 1 reflective (zero-flux wall) */
  double dt;     /* s */
  double a;      /* lattice spacing */
  double alpha;  /* in (0,1] */
} lpco_config;

typedef struct lpco_state {
  lpco_config c;
  int64_t n;       /* sites */
  int n_moments;   /* 0 or 3 */
  uint8_t *blocked;
  double *dF;
  double *link;    /* O10: 3n link factors or NULL; link[d*n + i] belongs to the link between i and i + e_d */
  double *pi;      /* O1 */
  double Zpart;    /* sum_j exp(-dF_j) */
  double *p_in[6]; /* p(nb_k(i) -> i), k = 2*d + (s>0) */
  double *stay;    /* O4 */
  double *cs, *sn; /* cos, sin of omega_i dt */
  double *g_re, *g_im, *t_re, *t_im; /* state and scratch */
  double *P[3], *Pt[3], *u[3];       /* moment fields, scratch, next-hop displacement */
  /* series */
  int64_t cap, steps;
  double *G;       /* 2*(cap+1): re, im */
  double *sabs;    /* cap+1 : sum_i |g_i(n)|  (tolerance scale) */
  double *Zd;      /* 3*(cap+2): Z_d[m] stored at [d*(cap+2) + m], m = 1..steps+1 */
} lpco_state;

/* ---- compensated summation (Neumaier) ---------------------------------- */
typedef struct { double s, c; } nsum;
static inline void ns_add(nsum *a, double x) {
  double t = a->s + x;
  if (fabs(a->s) >= fabs(x)) a->c += (a->s - t) + x; else a->c += (x - t) + a->s;
  a->s = t;
}
static inline double ns_val(const nsum *a) { return a->s + a->c; }

/* ---- O2: neighbour of site i along axis d in direction s = +-1 ---------
 * Periodic axis: wrap modulo n.  Reflective axis: out of range -> none (-1). */
static inline int64_t nb_xyz(const lpco_config *c, int64_t x, int64_t y, int64_t z, int d, int s) {
  int64_t n[3] = {c->nx, c->ny, c->nz};
  int64_t q[3] = {x, y, z};
  int64_t v = q[d] + s;
  if (v < 0 || v >= n[d]) {
    if (c->bc[d] != 0) return -1;
    v = (v + n[d]) % n[d];
  }
  q[d] = v;
  return (q[0] * n[1] + q[1]) * n[2] + q[2];
}
int64_t lpco_neighbor(const lpco_config *c, int64_t i, int d, int s) {
  int64_t z = i % c->nz;
  int64_t y = (i / c->nz) % c->ny;
  int64_t x = i / ((int64_t)c->nz * c->ny);
  return nb_xyz(c, x, y, z, d, s);
}

/* ---- O3: hop probability p(i->j), Eq. 1 with z = 6 and alpha ------------
 * 0 if there is no j, or either end is an obstacle.          */
double lpco_hop(const lpco_config *c, const double *dF, const uint8_t *blocked,
                int64_t i, int64_t j) {
  if (j < 0) return 0.0;
  if (blocked[i] || blocked[j]) return 0.0;
  double acc = (dF[j] > dF[i]) ? exp(-(dF[j] - dF[i])) : 1.0;
  return (c->alpha / 6.0) * acc;
}

/* ---- O10: per-link mobility factor alpha_ij ---------------
 * "a factor alpha_ij can be defined for each link between neighboring lattice sites i and j ... if the
 * probability of jumping from site i to site j is reduced, the probability of jumping from j to i must be
 * reduced by the same factor".  One number per link, stored at its lower end: link[d*n + i] is the factor of
 * the link between i and nb(i, d, +1), whichever way it is crossed.  j = nb(i, d, s).  No array: 1.      */
static double link_alpha(const double *link, int64_t n, int64_t i, int64_t j, int d, int s) {
  if (!link || j < 0) return 1.0;
  return (s > 0) ? link[(int64_t)d * n + i] : link[(int64_t)d * n + j];
}

static const int K_D[6] = {0, 0, 1, 1, 2, 2};
static const int K_S[6] = {-1, +1, -1, +1, -1, +1};

static double *dalloc(int64_t n) { return (double *)calloc((size_t)(n > 0 ? n : 1), sizeof(double)); }

void lpco_destroy(lpco_state *st) {
  if (!st) return;
  free(st->blocked); free(st->dF); free(st->link); free(st->pi); free(st->stay); free(st->cs); free(st->sn);
  for (int k = 0; k < 6; ++k) free(st->p_in[k]);
  free(st->g_re); free(st->g_im); free(st->t_re); free(st->t_im);
  for (int d = 0; d < 3; ++d) { free(st->P[d]); free(st->Pt[d]); free(st->u[d]); }
  free(st->G); free(st->sabs); free(st->Zd);
  free(st);
}

static void record_G(lpco_state *st, int64_t slot) {
  /* O6: G[n] = sum_i g_i(n), Eq. 12; also sum_i |g_i| for the tolerance scale. */
  const int64_t plane = (int64_t)st->c.ny * st->c.nz;
  const int nx = st->c.nx;
  double *pr = dalloc(nx), *pc = dalloc(nx), *qr = dalloc(nx), *qc = dalloc(nx), *ar = dalloc(nx), *ac = dalloc(nx);
#pragma omp parallel for schedule(static)
  for (int x = 0; x < nx; ++x) {
    nsum sr = {0, 0}, si = {0, 0}, sa = {0, 0};
    for (int64_t i = x * plane; i < (x + 1) * plane; ++i) {
      ns_add(&sr, st->g_re[i]);
      ns_add(&si, st->g_im[i]);
      ns_add(&sa, hypot(st->g_re[i], st->g_im[i]));
    }
    pr[x] = sr.s; pc[x] = sr.c; qr[x] = si.s; qc[x] = si.c; ar[x] = sa.s; ac[x] = sa.c;
  }
  nsum tr = {0, 0}, ti = {0, 0}, ta = {0, 0};
  for (int x = 0; x < nx; ++x) {
    ns_add(&tr, pr[x]); ns_add(&tr, pc[x]);
    ns_add(&ti, qr[x]); ns_add(&ti, qc[x]);
    ns_add(&ta, ar[x]); ns_add(&ta, ac[x]);
  }
  st->G[2 * slot] = ns_val(&tr);
  st->G[2 * slot + 1] = ns_val(&ti);
  st->sabs[slot] = ns_val(&ta);
  free(pr); free(pc); free(qr); free(qc); free(ar); free(ac);
}

static double plane_sum_prod(const lpco_state *st, const double *a, const double *b) {
  /* sum_i a_i * b_i (b may be NULL -> sum a_i), plane partials in x order. */
  const int64_t plane = (int64_t)st->c.ny * st->c.nz;
  const int nx = st->c.nx;
  double *ps = dalloc(nx), *pc = dalloc(nx);
#pragma omp parallel for schedule(static)
  for (int x = 0; x < nx; ++x) {
    nsum s = {0, 0};
    for (int64_t i = x * plane; i < (x + 1) * plane; ++i) ns_add(&s, b ? a[i] * b[i] : a[i]);
    ps[x] = s.s; pc[x] = s.c;
  }
  nsum t = {0, 0};
  for (int x = 0; x < nx; ++x) { ns_add(&t, ps[x]); ns_add(&t, pc[x]); }
  free(ps); free(pc);
  return ns_val(&t);
}

lpco_state *lpco_create_links(const lpco_config *c, const double *dF, const uint8_t *blocked,
                              const double *omega, const double *link, int n_moments, int64_t max_steps) {
  if (!c || !dF || !blocked || !omega) return NULL;
  if (c->nx < 1 || c->ny < 1 || c->nz < 1) return NULL;
  if (!(c->alpha > 0.0 && c->alpha <= 1.0)) return NULL;
  if (n_moments != 0 && n_moments != 3) return NULL;
  if (max_steps < 0) return NULL;
  lpco_state *st = (lpco_state *)calloc(1, sizeof(lpco_state));
  st->c = *c;
  const int64_t n = (int64_t)c->nx * c->ny * c->nz;
  st->n = n;
  st->n_moments = n_moments;
  st->cap = max_steps;
  st->blocked = (uint8_t *)malloc((size_t)n);
  memcpy(st->blocked, blocked, (size_t)n);
  st->dF = dalloc(n);
  memcpy(st->dF, dF, (size_t)n * sizeof(double));
  if (link) {
    for (int64_t k = 0; k < 3 * n; ++k)
      if (!(link[k] >= 0.0 && link[k] <= 1.0)) { lpco_destroy(st); return NULL; }
    st->link = dalloc(3 * n);
    memcpy(st->link, link, (size_t)(3 * n) * sizeof(double));
  }
  st->pi = dalloc(n); st->stay = dalloc(n); st->cs = dalloc(n); st->sn = dalloc(n);
  for (int k = 0; k < 6; ++k) st->p_in[k] = dalloc(n);
  st->g_re = dalloc(n); st->g_im = dalloc(n); st->t_re = dalloc(n); st->t_im = dalloc(n);
  st->G = dalloc(2 * (max_steps + 1)); st->sabs = dalloc(max_steps + 1);
  st->Zd = dalloc(3 * (max_steps + 2));

  /* O1: e_i = blocked ? 0 : exp(-dF_i);  Z = sum e_i;  pi_i = e_i / Z   (Eq. 2) */
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) st->pi[i] = blocked[i] ? 0.0 : exp(-dF[i]);
  st->Zpart = plane_sum_prod(st, st->pi, NULL);
  if (!(st->Zpart > 0.0) || !isfinite(st->Zpart)) { lpco_destroy(st); return NULL; }
  const double Z = st->Zpart;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) st->pi[i] = st->pi[i] / Z;

  /* O3, O4 tables and the Eq. 13 phase factor exp(i omega_i dt) (Q2, Q4). */
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < n; ++i) {
    double out = 0.0;
    for (int k = 0; k < 6; ++k) {
      int64_t j = lpco_neighbor(c, i, K_D[k], K_S[k]);
      const double aij = link_alpha(st->link, n, i, j, K_D[k], K_S[k]);   /* O10: same factor both ways */
      st->p_in[k][i] = (j < 0) ? 0.0 : aij * lpco_hop(c, dF, blocked, j, i);
      out += aij * lpco_hop(c, dF, blocked, i, j);
    }
    st->stay[i] = 1.0 - out;
    st->cs[i] = cos(omega[i] * c->dt);
    st->sn[i] = sin(omega[i] * c->dt);
  }

  /* g(0) = pi (real): G[0] = 1 (Q9, Q10). */
  memcpy(st->g_re, st->pi, (size_t)n * sizeof(double));
  record_G(st, 0);

  if (n_moments == 3) {
    for (int d = 0; d < 3; ++d) { st->P[d] = dalloc(n); st->Pt[d] = dalloc(n); st->u[d] = dalloc(n); }
    /* O7 */
    double *z1 = dalloc(n);
    for (int d = 0; d < 3; ++d) {
#pragma omp parallel for schedule(static)
      for (int64_t i = 0; i < n; ++i) {
        double P1 = 0.0, ui = 0.0, m2 = 0.0;
        for (int s = -1; s <= 1; s += 2) {
          int64_t j = lpco_neighbor(c, i, d, s);
          if (j < 0) continue;
          /* arrival at i from j = i + s e_d: displacement -s a */
          const double aij = link_alpha(st->link, n, i, j, d, s);
          P1 += st->pi[j] * (aij * lpco_hop(c, dF, blocked, j, i)) * (-(double)s * c->a);
          double po = aij * lpco_hop(c, dF, blocked, i, j);
          ui += po * ((double)s * c->a);
          m2 += po * c->a * c->a;
        }
        st->P[d][i] = P1;
        st->u[d][i] = ui;
        z1[i] = st->pi[i] * m2;
      }
      st->Zd[d * (st->cap + 2) + 1] = plane_sum_prod(st, z1, NULL);
    }
    free(z1);
  }
  st->steps = 0;
  return st;
}

lpco_state *lpco_create(const lpco_config *c, const double *dF, const uint8_t *blocked,
                        const double *omega, int n_moments, int64_t max_steps) {
  return lpco_create_links(c, dF, blocked, omega, NULL, n_moments, max_steps);
}

/* O5 for a real field (no phase): out_i = stay_i f_i + sum_k p_in[k][i] f_{nb_k(i)} */
static void propagate_real(const lpco_state *st, const double *f, double *out) {
  const lpco_config *c = &st->c;
#pragma omp parallel for schedule(static)
  for (int64_t x = 0; x < c->nx; ++x)
    for (int64_t y = 0; y < c->ny; ++y)
      for (int64_t z = 0; z < c->nz; ++z) {
        const int64_t i = (x * c->ny + y) * c->nz + z;
        if (st->blocked[i]) { out[i] = 0.0; continue; }
        double acc = st->stay[i] * f[i];
        for (int k = 0; k < 6; ++k) {
          int64_t j = nb_xyz(c, x, y, z, K_D[k], K_S[k]);
          if (j >= 0) acc += st->p_in[k][i] * f[j];
        }
        out[i] = acc;
      }
}

/* One propagation step: O8 (moments) then O5/O6 (magnetisation). */
static void step_once(lpco_state *st) {
  const lpco_config *c = &st->c;
  if (st->n_moments == 3) {
    for (int d = 0; d < 3; ++d) {
      /* Z_d[k+1] = sum_i P^d_i(k) u^d_i with k = steps+1 */
      st->Zd[d * (st->cap + 2) + st->steps + 2] = plane_sum_prod(st, st->P[d], st->u[d]);
      propagate_real(st, st->P[d], st->Pt[d]);
      double *t = st->P[d]; st->P[d] = st->Pt[d]; st->Pt[d] = t;
    }
  }
#pragma omp parallel for schedule(static)
  for (int64_t x = 0; x < c->nx; ++x)
    for (int64_t y = 0; y < c->ny; ++y)
      for (int64_t z = 0; z < c->nz; ++z) {
        const int64_t i = (x * c->ny + y) * c->nz + z;
        if (st->blocked[i]) { st->t_re[i] = 0.0; st->t_im[i] = 0.0; continue; }
        double ar = st->stay[i] * st->g_re[i];
        double ai = st->stay[i] * st->g_im[i];
        for (int k = 0; k < 6; ++k) {
          int64_t j = nb_xyz(c, x, y, z, K_D[k], K_S[k]);
          if (j >= 0) {
            ar += st->p_in[k][i] * st->g_re[j];
            ai += st->p_in[k][i] * st->g_im[j];
          }
        }
        /* (cos + i sin)(ar + i ai) */
        st->t_re[i] = st->cs[i] * ar - st->sn[i] * ai;
        st->t_im[i] = st->cs[i] * ai + st->sn[i] * ar;
      }
  double *t;
  t = st->g_re; st->g_re = st->t_re; st->t_re = t;
  t = st->g_im; st->g_im = st->t_im; st->t_im = t;
  st->steps += 1;
  record_G(st, st->steps);
}

int lpco_step(lpco_state *st, int64_t n) {
  if (!st || n < 0 || st->steps + n > st->cap) return -1;
  for (int64_t k = 0; k < n; ++k) step_once(st);
  return 0;
}

/* Arbitrary initial magnetisation (interleaved re,im); resets the series. Blocked sites -> 0. */
int lpco_set_g(lpco_state *st, const double *re_im) {
  if (!st || !re_im) return -1;
  for (int64_t i = 0; i < st->n; ++i) {
    st->g_re[i] = st->blocked[i] ? 0.0 : re_im[2 * i];
    st->g_im[i] = st->blocked[i] ? 0.0 : re_im[2 * i + 1];
  }
  st->steps = 0;
  record_G(st, 0);
  return 0;
}

/* Real-field propagation of an arbitrary density (equilibration / relaxation tests). */
int lpco_propagate_real(const lpco_state *st, const double *rho_in, double *rho_out, int64_t n_steps) {
  if (!st || !rho_in || !rho_out || n_steps < 0) return -1;
  double *a = dalloc(st->n), *b = dalloc(st->n);
  for (int64_t i = 0; i < st->n; ++i) a[i] = st->blocked[i] ? 0.0 : rho_in[i];
  for (int64_t k = 0; k < n_steps; ++k) { propagate_real(st, a, b); double *t = a; a = b; b = t; }
  memcpy(rho_out, a, (size_t)st->n * sizeof(double));
  free(a); free(b);
  return 0;
}

/* Equilibration loop of the paper's workflow (Fig. 3 step 3): iterate the
 * density update rho <- W rho and compare rho(t) with rho(t+1); stop when the difference falls below
 * `threshold` or after `max_iters` iterations.  The paper does not name the norm: DESIGN.md reading
 * Q25 takes the largest per-site change, delta(t+1) = max_i |rho_i(t+1) - rho_i(t)|, and stops as soon
 * as delta < threshold (the updated density is kept).  deltas_out (may be NULL) receives
 * delta(1..iters).  Returns the number of iterations done, or -1 on bad arguments. */
int64_t lpco_equilibrate(const lpco_state *st, double *rho_inout, double threshold, int64_t max_iters, double *deltas_out) {
  if (!st || !rho_inout || max_iters < 0) return -1;
  double *a = dalloc(st->n), *b = dalloc(st->n);
  for (int64_t i = 0; i < st->n; ++i) a[i] = st->blocked[i] ? 0.0 : rho_inout[i];
  int64_t it = 0;
  while (it < max_iters) {
    propagate_real(st, a, b);
    double delta = 0.0;
    for (int64_t i = 0; i < st->n; ++i) {
      const double d = fabs(b[i] - a[i]);
      if (d > delta) delta = d;
    }
    double *t = a; a = b; b = t;
    if (deltas_out) deltas_out[it] = delta;
    ++it;
    if (delta < threshold) break;
  }
  memcpy(rho_inout, a, (size_t)st->n * sizeof(double));
  free(a); free(b);
  return it;
}

/* ---- read-outs ----------------------------------------------------------- */
int64_t lpco_steps(const lpco_state *st) { return st->steps; }
double lpco_partition_sum(const lpco_state *st) { return st->Zpart; }
void lpco_get_pi(const lpco_state *st, double *out) { memcpy(out, st->pi, (size_t)st->n * sizeof(double)); }
void lpco_get_stay(const lpco_state *st, double *out) { memcpy(out, st->stay, (size_t)st->n * sizeof(double)); }
void lpco_get_p_in(const lpco_state *st, int k, double *out) { memcpy(out, st->p_in[k], (size_t)st->n * sizeof(double)); }
void lpco_get_g(const lpco_state *st, double *re_im) {
  for (int64_t i = 0; i < st->n; ++i) { re_im[2 * i] = st->g_re[i]; re_im[2 * i + 1] = st->g_im[i]; }
}
int lpco_get_P(const lpco_state *st, int d, double *out) {
  if (st->n_moments != 3) return -1;
  memcpy(out, st->P[d], (size_t)st->n * sizeof(double));
  return 0;
}
int lpco_get_u(const lpco_state *st, int d, double *out) {
  if (st->n_moments != 3) return -1;
  memcpy(out, st->u[d], (size_t)st->n * sizeof(double));
  return 0;
}
/* G[first .. first+count) as interleaved re,im; sabs the matching sum_i |g_i|. */
int lpco_get_fid(const lpco_state *st, int64_t first, int64_t count, double *out_re_im, double *out_sabs) {
  if (first < 0 || count < 0 || first + count > st->steps + 1) return -1;
  memcpy(out_re_im, st->G + 2 * first, (size_t)(2 * count) * sizeof(double));
  if (out_sabs) memcpy(out_sabs, st->sabs + first, (size_t)count * sizeof(double));
  return 0;
}
/* Z_d[1..count] into vacf[d*count + (m-1)] and D_d from those (O8):
 *   D_d = Z_d[1]/(2 dt) + (1/dt) sum_{m=2..count} Z_d[m]                    */
int lpco_get_moments(const lpco_state *st, int64_t count, double *vacf, double *D) {
  if (st->n_moments != 3 || count < 1 || count > st->steps + 1) return -1;
  for (int d = 0; d < 3; ++d) {
    const double *z = st->Zd + d * (st->cap + 2);
    nsum s = {0, 0};
    for (int64_t m = 1; m <= count; ++m) {
      vacf[d * count + (m - 1)] = z[m];
      if (m >= 2) ns_add(&s, z[m]);
    }
    D[d] = z[1] / (2.0 * st->c.dt) + ns_val(&s) / st->c.dt;
  }
  return 0;
}
