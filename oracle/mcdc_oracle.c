/* mcdc_oracle.c — TEST INFRASTRUCTURE ONLY (see mcdc_oracle.h).
 *
 * Plain single-threaded C oracle of the multigroup time-dependent Monte Carlo
 * history loop (§2 "history-based algorithm"; §3
 * fixed source, multigroup physics, mesh tallies, time census, population
 * control).  The paper gives no equations: each function cites the DESIGN.md §3
 * reading (R-numbers; identical to SURVEY.md §8(c)) it follows.
 *
 * Build: gcc -std=c11 -O2 -ffp-contract=off -fPIC -shared  (no libm in the
 * transport path; only IEEE +,-,*,/,sqrt,fma which round identically anywhere).
 */
#include "mcdc_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ */
/* R1 (C.1) Philox4x32-10: round = two 32x32->64 multiplies, xor with  */
/* key, key bumped by Weyl constants between rounds.                   */
/* ------------------------------------------------------------------ */
void oracle_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4])
{
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R1 (C.1): 52-bit integer k = (hi<<20)|(lo>>12); xi = (k + 0.5) * 2^-52,
 * exact in binary64, never 0 or 1. */
double oracle_uniform52(uint32_t hi, uint32_t lo)
{
  uint64_t k = ((uint64_t)hi << 20) | (uint64_t)(lo >> 12);
  return ((double)k + 0.5) * 0x1.0p-52;
}

/* purpose (block) codes, R1 */
enum { B_SRC_XY = 0, B_SRC_ZG = 1, B_SRC_DIR = 2, B_SRC_PIN = 3, B_DCOL = 4,
       B_REACT = 5, B_SCAT_DIR = 6, B_FIS_N = 7, B_ROULETTE = 8, B_DELAY = 9, B_SRC_TIME = 10, B_CHILD = 0x100, B_FPRINT = 0x200 };

typedef struct { double a, b; uint32_t r0, r1; } draw2;

/* key = pid, counter = (ectr, block, seedb_lo, seedb_hi) */
static draw2 draw(uint64_t pid, uint32_t ectr, uint32_t block, uint64_t seedb)
{
  uint32_t key[2] = { (uint32_t)pid, (uint32_t)(pid >> 32) };
  uint32_t ctr[4] = { ectr, block, (uint32_t)seedb, (uint32_t)(seedb >> 32) };
  uint32_t o[4];
  oracle_philox4x32_10(key, ctr, o);
  draw2 d;
  d.a = oracle_uniform52(o[0], o[1]);
  d.b = oracle_uniform52(o[2], o[3]);
  d.r0 = o[0]; d.r1 = o[1];
  return d;
}

/* ------------------------------------------------------------------ */
/* R2 (C.2, App. B) math functions: IEEE ops + explicit fma only.      */
/* ------------------------------------------------------------------ */
double oracle_log(double x)
{
  /* x normal, in (0,1]. split x = m * 2^e, m in [1,2) */
  uint64_t bits; memcpy(&bits, &x, 8);
  int e = (int)((bits >> 52) & 0x7FF) - 1023;
  bits = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FF0000000000000ull;
  double m; memcpy(&m, &bits, 8);
  const double SQRT2 = 0x1.6a09e667f3bcdp+0; /* nearest double to sqrt 2 */
  if (m > SQRT2) { m = m * 0.5; e += 1; }
  double f = m - 1.0;
  double s = f / (2.0 + f);
  double z = s * s;
  double P = 1.0 / 21.0;
  for (int n = 9; n >= 0; --n) P = fma(P, z, 1.0 / (double)(2 * n + 1));
  const double LN2 = 0x1.62e42fefa39efp-1;
  return fma((double)e, LN2, (s + s) * P);
}

void oracle_sincos2pi(double u, double *cc, double *ss)
{
  double q4 = 4.0 * u;
  int k = (int)q4; /* q4 in (0,4): truncation = floor, exact */
  double r = q4 - (double)k;
  int swap = 0;
  if (r > 0.5) { r = 1.0 - r; swap = 1; }
  const double HALF_PI = 0x1.921fb54442d18p+0;
  double th = r * HALF_PI;
  double z = th * th;
  /* factorials exact in binary64 up to 18! */
  double fact[18]; fact[0] = 1.0;
  for (int n = 1; n < 18; ++n) fact[n] = fact[n - 1] * (double)n;
  /* sin: theta * sum_{n=0..7} (-1)^n z^n/(2n+1)!   cos: sum_{n=0..8} (-1)^n z^n/(2n)! */
  double S = -1.0 / fact[15];
  for (int n = 6; n >= 0; --n) {
    double c = 1.0 / fact[2 * n + 1];
    if (n & 1) c = -c;
    S = fma(S, z, c);
  }
  S = th * S;
  double C = 1.0 / fact[16];
  for (int n = 7; n >= 0; --n) {
    double c = 1.0 / fact[2 * n];
    if (n & 1) c = -c;
    C = fma(C, z, c);
  }
  if (swap) { double t = S; S = C; C = t; }
  switch (k & 3) {
    case 0: *cc = C;  *ss = S;  break;
    case 1: *cc = -S; *ss = C;  break;
    case 2: *cc = -C; *ss = -S; break;
    default: *cc = S; *ss = -C; break;
  }
}

/* ------------------------------------------------------------------ */
/* Problem record and set-up, R3 (C.3)                                  */
/* ------------------------------------------------------------------ */
typedef struct {
  double x, y, z, t, ux, uy, uz, w;
  uint64_t pid;
  uint32_t ectr;
  int32_t g, ix, iy, iz, inside;
  int32_t reg;                      /* C.18: region of the quadric CSG the particle is in (-1: none) */
} particle;

typedef struct { particle *v; size_t n, cap; } bank;

struct oracle_problem {
  int32_t M, G;
  double *sigma_t, *sigma_c, *sigma_f, *nu, *sigma_s, *chi, *speed;
  double *sigma_s_row; /* [M][G]    sum over g' ascending */
  double *cdf_s;       /* [M][G][G] */
  double *cdf_chi;     /* [M][G]    */
  double *cdf_src;     /* [G]       */
  int32_t nx, ny, nz;
  double *xs, *ys, *zs;
  int32_t *mat_outer, *mat_inner;
  double *radius;
  int32_t bc[6];
  int32_t src_kind, src_isotropic;
  double src_lo[3], src_hi[3], src_dir[3], src_t0;
  int64_t n_pins; int32_t *pin_cell; /* row-major list of cells with mat_inner>=0 */
  int32_t tnx, tny, tnz, tnt;
  double *txs, *tys, *tzs, *tts;
  int32_t n_census; double *t_census; uint64_t comb_target;
  int32_t time_crossing;
  /* results */
  size_t n_track;                   /* bins of the track-length block */
  size_t n_tally;                   /* all bins: n_track, or 2 n_track with the time-crossing block */
  double *tally, *tally_comp;       /* current batch: sum and Neumaier compensation */
  double *sum1, *sum2;              /* over batches of per-batch raw tallies */
  uint32_t n_batch_done; uint64_t n_hist_per_batch;
  uint64_t *counters;               /* [batch][step][16] */
  uint32_t n_steps;
  /* k-eigenvalue mode (DESIGN.md section 3 C.14): one "step" = one fission generation */
  int32_t eig_inactive, eig_active; /* both 0: fixed-source mode */
  double eig_k0;
  double *k_cycle;                  /* [batch][cycle] generation estimate k_c N_f / N of every cycle */
  double cur_k;                     /* k the running cycle normalises its fission yield with (0: fixed source) */
  int cur_score;                    /* the running cycle scores the tally (active cycle / fixed source) */
  /* implicit capture, weight roulette and the weighted comb (PAPER.md:83 "implicit capture", :59
   * "population control techniques [9,10]"; DESIGN.md section 3 C.15) */
  int ic_on; double ic_w_roulette, ic_w_survive;
  /* delayed neutrons (PAPER.md:105 "delayed neutron precursor", :119; DESIGN.md section 3 C.16) */
  /* source with a time extent ("making the specified source active only in the first fifty
   * seconds"; DESIGN.md section 3 C.17): birth time uniform in [src_t0, src_t1]; src_t1 <= src_t0: pulse */
  double src_t1;
  int dn_J;                          /* precursor groups; 0: every fission neutron is prompt */
  double *dn_nu;                     /* [n_mat][G][J] delayed yield per fission and precursor group */
  double *dn_nu_prompt;              /* [n_mat][G] nu - sum_j dn_nu (ascending sum) */
  double *dn_lambda;                 /* [n_mat][J] decay constants */
  double *dn_cdf_chi;                /* [n_mat][J][G] CDF of the delayed emission spectra */
  /* quadric-surface CSG (DESIGN.md section 3 C.18) and moving surfaces (C.19) */
  int32_t csg_n_surf, csg_n_region;  /* 0: lattice geometry */
  double *csg_coef;                  /* [n_surf][10] A B C D E F G H J K */
  int32_t *csg_rsurf;                /* [n_region][8] signed surface ids + 1, 0-terminated */
  int32_t *csg_rmat;                 /* [n_region] */
  int32_t mv_n_tau;                  /* 0: all surfaces at rest */
  double *mv_tau;                    /* [n_tau] break times */
  double *mv_disp;                   /* [n_surf][n_tau][3] displacement at the break times */
  double *mv_vel;                    /* [n_surf][n_tau][3] velocity in [tau_k, tau_k+1) (0 in the last entry) */
};

static void *dup_mem(const void *src, size_t bytes)
{
  void *p = malloc(bytes ? bytes : 1);
  if (p && src && bytes) memcpy(p, src, bytes);
  return p;
}

/* running sum ascending, one divide per entry, last forced to 1.0 (R3) */
static void make_cdf(const double *pdf, int n, double total, double *cdf)
{
  double run = 0.0;
  for (int j = 0; j < n; ++j) { run = run + pdf[j]; cdf[j] = (total > 0.0) ? run / total : 0.0; }
  cdf[n - 1] = 1.0;
}

static int ascending(const double *p, int n1)
{
  for (int i = 0; i + 1 < n1; ++i) if (!(p[i] < p[i + 1])) return 0;
  return 1;
}

int oracle_create(const oracle_input *in, oracle_problem **out)
{
  if (!in || !out) return 1;
  const int M = in->n_mat, G = in->n_group;
  if (M < 1 || G < 1 || G > 255 || in->nx < 1 || in->ny < 1 || in->nz < 1) return 1;
  if (in->nx > 1023 || in->ny > 1023 || in->nz > 1023) return 1;
  if (in->tnx < 1 || in->tny < 1 || in->tnz < 1 || in->tnt < 1) return 1;
  if (!ascending(in->xs, in->nx + 1) || !ascending(in->ys, in->ny + 1) ||
      !ascending(in->zs, in->nz + 1)) return 1;
  if (!ascending(in->txs, in->tnx + 1) || !ascending(in->tys, in->tny + 1) ||
      !ascending(in->tzs, in->tnz + 1) || !ascending(in->tts, in->tnt + 1)) return 1;
  /* tally mesh covers the geometry box */
  if (in->txs[0] > in->xs[0] || in->txs[in->tnx] < in->xs[in->nx]) return 1;
  if (in->tys[0] > in->ys[0] || in->tys[in->tny] < in->ys[in->ny]) return 1;
  if (in->tzs[0] > in->zs[0] || in->tzs[in->tnz] < in->zs[in->nz]) return 1;
  if (in->n_census < 0) return 1;
  if (in->n_census > 0 && !ascending(in->t_census, in->n_census)) return 1;
  for (int k = 0; k < in->n_census; ++k) { /* every census time is a tally time edge, bit for bit */
    int found = 0;
    for (int j = 0; j <= in->tnt; ++j) if (in->tts[j] == in->t_census[k]) found = 1;
    if (!found) return 1;
  }
  if (in->tts[0] > in->src_t0) return 1;

  oracle_problem *p = (oracle_problem *)calloc(1, sizeof *p);
  if (!p) return 2;
  p->M = M; p->G = G;
  p->sigma_t = dup_mem(in->sigma_t, sizeof(double) * M * G);
  p->sigma_c = dup_mem(in->sigma_c, sizeof(double) * M * G);
  p->sigma_f = dup_mem(in->sigma_f, sizeof(double) * M * G);
  p->nu      = dup_mem(in->nu,      sizeof(double) * M * G);
  p->chi     = dup_mem(in->chi,     sizeof(double) * M * G);
  p->sigma_s = dup_mem(in->sigma_s, sizeof(double) * M * G * G);
  p->speed   = dup_mem(in->speed,   sizeof(double) * G);
  p->sigma_s_row = malloc(sizeof(double) * M * G);
  p->cdf_s   = malloc(sizeof(double) * M * G * G);
  p->cdf_chi = malloc(sizeof(double) * M * G);
  p->cdf_src = malloc(sizeof(double) * G);
  int bad = 0;
  for (int m = 0; m < M; ++m) {
    for (int g = 0; g < G; ++g) {
      const double *row = p->sigma_s + ((size_t)m * G + g) * G;
      double sr = 0.0;
      for (int j = 0; j < G; ++j) { if (row[j] < 0.0) bad = 1; sr = sr + row[j]; }
      p->sigma_s_row[m * G + g] = sr;
      make_cdf(row, G, sr, p->cdf_s + ((size_t)m * G + g) * G);
      double st = p->sigma_t[m * G + g];
      if (!(st > 0.0)) bad = 1;
      double tot = sr + p->sigma_c[m * G + g] + p->sigma_f[m * G + g];
      if (fabs(st - tot) > 1e-12 * st) bad = 1;
      if (p->sigma_c[m * G + g] < 0.0 || p->sigma_f[m * G + g] < 0.0) bad = 1;
    }
    double cs = 0.0;
    for (int g = 0; g < G; ++g) cs = cs + p->chi[m * G + g];
    int fissile = 0;
    for (int g = 0; g < G; ++g) if (p->sigma_f[m * G + g] > 0.0) fissile = 1;
    if (fissile && fabs(cs - 1.0) > 1e-12) bad = 1;
    make_cdf(p->chi + m * G, G, cs, p->cdf_chi + m * G);
  }
  for (int g = 0; g < G; ++g) if (!(p->speed[g] > 0.0)) bad = 1;
  {
    double ps = 0.0;
    for (int g = 0; g < G; ++g) ps = ps + in->src_group_pdf[g];
    if (fabs(ps - 1.0) > 1e-12) bad = 1;
    make_cdf(in->src_group_pdf, G, ps, p->cdf_src);
  }
  p->nx = in->nx; p->ny = in->ny; p->nz = in->nz;
  size_t nc = (size_t)in->nx * in->ny * in->nz;
  p->xs = dup_mem(in->xs, sizeof(double) * (in->nx + 1));
  p->ys = dup_mem(in->ys, sizeof(double) * (in->ny + 1));
  p->zs = dup_mem(in->zs, sizeof(double) * (in->nz + 1));
  p->mat_outer = dup_mem(in->mat_outer, sizeof(int32_t) * nc);
  p->mat_inner = dup_mem(in->mat_inner, sizeof(int32_t) * nc);
  p->radius = dup_mem(in->radius, sizeof(double) * nc);
  memcpy(p->bc, in->bc, sizeof p->bc);
  p->pin_cell = malloc(sizeof(int32_t) * nc);
  p->n_pins = 0;
  for (size_t c = 0; c < nc; ++c) {
    if (p->mat_outer[c] < 0 || p->mat_outer[c] >= M) bad = 1;
    if (p->mat_inner[c] >= M) bad = 1;
    if (p->mat_inner[c] >= 0) {
      int ix = (int)(c % in->nx), iy = (int)((c / in->nx) % in->ny);
      double hw = 0.5 * (p->xs[ix + 1] - p->xs[ix]), hh = 0.5 * (p->ys[iy + 1] - p->ys[iy]);
      if (!(p->radius[c] > 0.0) || !(p->radius[c] < hw) || !(p->radius[c] < hh)) bad = 1;
      p->pin_cell[p->n_pins++] = (int32_t)c;
    }
  }
  p->src_kind = in->src_kind; p->src_isotropic = in->src_isotropic; p->src_t0 = in->src_t0; p->src_t1 = in->src_t0;
  memcpy(p->src_lo, in->src_lo, sizeof p->src_lo);
  memcpy(p->src_hi, in->src_hi, sizeof p->src_hi);
  memcpy(p->src_dir, in->src_dir, sizeof p->src_dir);
  if (p->src_kind < 0 || p->src_kind > 3) bad = 1;   /* (kind 3 needs oracle_set_csg: checked at run) */
  if (p->src_kind == 2 && p->n_pins == 0) bad = 1;
  p->tnx = in->tnx; p->tny = in->tny; p->tnz = in->tnz; p->tnt = in->tnt;
  p->txs = dup_mem(in->txs, sizeof(double) * (in->tnx + 1));
  p->tys = dup_mem(in->tys, sizeof(double) * (in->tny + 1));
  p->tzs = dup_mem(in->tzs, sizeof(double) * (in->tnz + 1));
  p->tts = dup_mem(in->tts, sizeof(double) * (in->tnt + 1));
  p->n_census = in->n_census;
  p->t_census = dup_mem(in->t_census, sizeof(double) * (in->n_census > 0 ? in->n_census : 1));
  p->comb_target = in->comb_target;
  p->n_steps = in->n_census > 0 ? (uint32_t)in->n_census : 1u;
  p->time_crossing = in->time_crossing != 0;
  p->n_track = (size_t)in->tnt * G * in->tnz * in->tny * in->tnx;
  p->n_tally = p->n_track * (p->time_crossing ? 2 : 1);
  p->tally = calloc(p->n_tally, sizeof(double));
  p->tally_comp = calloc(p->n_tally, sizeof(double));
  p->sum1 = calloc(p->n_tally, sizeof(double));
  p->sum2 = calloc(p->n_tally, sizeof(double));
  if (bad) { oracle_destroy(p); return 1; }
  *out = p;
  return 0;
}

void oracle_destroy(oracle_problem *p)
{
  if (p) { free(p->k_cycle); free(p->dn_nu); free(p->dn_nu_prompt); free(p->dn_lambda); free(p->dn_cdf_chi);
           free(p->csg_coef); free(p->csg_rsurf); free(p->csg_rmat); free(p->mv_tau); free(p->mv_disp); free(p->mv_vel); }
  if (!p) return;
  free(p->sigma_t); free(p->sigma_c); free(p->sigma_f); free(p->nu); free(p->sigma_s);
  free(p->chi); free(p->speed); free(p->sigma_s_row); free(p->cdf_s); free(p->cdf_chi);
  free(p->cdf_src); free(p->xs); free(p->ys); free(p->zs); free(p->mat_outer);
  free(p->mat_inner); free(p->radius); free(p->pin_cell); free(p->txs); free(p->tys);
  free(p->tzs); free(p->tts); free(p->t_census); free(p->tally); free(p->tally_comp);
  free(p->sum1); free(p->sum2); free(p->counters);
  free(p);
}

/* ------------------------------------------------------------------ */
/* Geometry helpers, R4 (C.4) and App. C                                */
/* ------------------------------------------------------------------ */
#define INF ((double)INFINITY)

/* direction-aware lookup: largest i with planes[i] <= p; if planes[i]==p and
 * the particle moves down the axis, take the lower interval; clamp to [0,n-1] */
static int lookup(const double *planes, int n, double p, double u)
{
  int i = -1;
  for (int j = 0; j <= n; ++j) if (planes[j] <= p) i = j;
  if (i >= 0 && planes[i] == p && u < 0.0) i -= 1;
  if (i < 0) i = 0;
  if (i > n - 1) i = n - 1;
  return i;
}

/* App. C.1 cylinder: logical region flag selects the root; result clamped >= 0 */
double oracle_cyl_distance(double x, double y, double ux, double uy, double cx,
                           double cy, double R, int inside)
{
  double dx = x - cx, dy = y - cy;
  double A = fma(ux, ux, uy * uy);
  if (A == 0.0) return INF;
  double Bh = fma(dx, ux, dy * uy);
  double Cc = fma(dx, dx, dy * dy) - R * R;
  double D = fma(Bh, Bh, -(A * Cc));
  double s;
  if (inside) {
    if (D <= 0.0) D = 0.0;
    if (Bh <= 0.0) s = (sqrt(D) - Bh) / A;
    else           s = -Cc / (sqrt(D) + Bh);
    if (s < 0.0) s = 0.0;
    return s;
  }
  if (Bh >= 0.0 || D <= 0.0) return INF;
  s = Cc / (sqrt(D) - Bh);
  if (s < 0.0) s = 0.0;
  return s;
}

/* ---- C.18 quadric surfaces.  Plain IEEE expressions, evaluated left to right as written (no fma). ---- */
static double quad_eval(const double *q, double x, double y, double z)
{
  return q[0] * x * x + q[1] * y * y + q[2] * z * z + q[3] * x * y + q[4] * y * z + q[5] * z * x +
         q[6] * x + q[7] * y + q[8] * z + q[9];
}

/* g(s) = sense f(r + s u) = a s^2 + 2 b s + c is positive on the particle's (logical) side; the distance is the
 * first s >= 0 at which g turns negative: the root (-b - sqrt(b^2 - a c)) / a, whatever the sign of a, written
 * without cancellation as c / (sqrt(D) - b) when b <= 0.  The side is logical, never re-derived from the
 * coordinates: a particle sitting on the surface it has just crossed (c = +-rounding) finds the far root or none. */
double oracle_quadric_distance(const double *q, double sense, double x, double y, double z,
                               double ux, double uy, double uz)
{
  const double a = sense * (q[0] * ux * ux + q[1] * uy * uy + q[2] * uz * uz + q[3] * ux * uy + q[4] * uy * uz + q[5] * uz * ux);
  const double b = sense * (q[0] * x * ux + q[1] * y * uy + q[2] * z * uz +
                            0.5 * (q[3] * (x * uy + y * ux) + q[4] * (y * uz + z * uy) + q[5] * (z * ux + x * uz) +
                                   q[6] * ux + q[7] * uy + q[8] * uz));
  const double c = sense * quad_eval(q, x, y, z);
  double s;
  if (a == 0.0) {
    if (!(b < 0.0)) return INF;
    s = c / (-2.0 * b);
  } else {
    double D = b * b - a * c;
    if (a > 0.0) {
      if (!(b < 0.0) || !(D > 0.0)) return INF;
      s = c / (sqrt(D) - b);
    } else {
      if (D < 0.0) D = 0.0;
      const double sq = sqrt(D);
      if (b <= 0.0) { const double den = sq - b; s = den > 0.0 ? c / den : 0.0; }
      else s = -(b + sq) / a;
    }
  }
  if (!(s >= 0.0)) s = 0.0;
  return s;
}

/* C.19: displacement of surface s at time t and its velocity there (piecewise linear through the break times) */
static void surf_motion(const oracle_problem *p, int s, double t, double d[3], double vel[3])
{
  d[0] = d[1] = d[2] = 0.0; vel[0] = vel[1] = vel[2] = 0.0;
  const int n = p->mv_n_tau;
  if (n == 0) return;
  int k = -1;
  for (int j = 0; j < n; ++j) if (p->mv_tau[j] <= t) k = j;
  const double *D = p->mv_disp + (size_t)s * n * 3, *V = p->mv_vel + (size_t)s * n * 3;
  if (k < 0) { d[0] = D[0]; d[1] = D[1]; d[2] = D[2]; return; }
  const double dt = t - p->mv_tau[k];
  for (int i = 0; i < 3; ++i) { vel[i] = V[k * 3 + i]; d[i] = D[k * 3 + i] + vel[i] * dt; }
}

/* sign of f_s at a point and time, from the coordinates (source lookup; surfaces a crossing does not involve) */
static int surf_side(const oracle_problem *p, int s, double x, double y, double z, double t)
{
  double d[3], vel[3];
  surf_motion(p, s, t, d, vel);
  return quad_eval(p->csg_coef + (size_t)s * 10, x - d[0], y - d[1], z - d[2]) > 0.0 ? 1 : -1;
}

/* region that holds the point: all sides from the coordinates (from < 0), or, after the particle of region
 * `from` has crossed surface `crossed`, the logical sides of `from` with that one flipped and coordinates only
 * for the surfaces `from` does not know.  First match in index order; -1: none. */
static int find_region(const oracle_problem *p, int from, int crossed, double x, double y, double z, double t)
{
  for (int q = 0; q < p->csg_n_region; ++q) {
    int ok = 1;
    for (int j = 0; j < 8 && ok; ++j) {
      const int e = p->csg_rsurf[q * 8 + j];
      if (e == 0) break;
      const int sf = (e > 0 ? e : -e) - 1, want = e > 0 ? 1 : -1;
      int have = 0;
      if (from >= 0)
        for (int i = 0; i < 8; ++i) {
          const int f = p->csg_rsurf[from * 8 + i];
          if (f == 0) break;
          if ((f > 0 ? f : -f) - 1 == sf) { have = f > 0 ? 1 : -1; if (sf == crossed) have = -have; break; }
        }
      if (have == 0) have = surf_side(p, sf, x, y, z, t);
      if (have != want) ok = 0;
    }
    if (ok) return q;
  }
  return -1;
}

static double plane_distance(const double *planes, int i, double p, double u)
{
  double d;
  if (u > 0.0)      d = (planes[i + 1] - p) / u;
  else if (u < 0.0) d = (planes[i] - p) / u;
  else return INF;
  if (d < 0.0) d = 0.0; /* C.5 step 4 clamp */
  return d;
}

/* App. C.2: distance along the flight to the next tally plane of one axis,
 * always recomputed from the flight origin; clamped >= 0 */
static double tally_s(const double *T, int j, double p, double u)
{
  double s;
  if (u > 0.0)      s = (T[j + 1] - p) / u;
  else if (u < 0.0) s = (T[j] - p) / u;
  else return INF;
  if (s < 0.0) s = 0.0;
  return s;
}
static double tally_st(const double *T, int j, double t, double v)
{
  double s = (T[j + 1] - t) * v;
  if (s < 0.0) s = 0.0;
  return s;
}

/* App. C.2 tally march.  Calls score(ctx, jt, jz, jy, jx, len) for every
 * sub-segment of positive length; returns their number, or -1 when an index
 * leaves the mesh. */
typedef void (*score_fn)(void *ctx, int jt, int jz, int jy, int jx, double len);

/* cross (may be NULL) is called when the march passes the upper time edge of bin jt, with the
 * spatial bin the particle is in at that moment; jend (may be NULL) receives the bins (t, z, y, x)
 * the flight ends in. */
static int64_t march_core(const double *txs, int32_t tnx, const double *tys, int32_t tny,
                          const double *tzs, int32_t tnz, const double *tts, int32_t tnt,
                          const double pos[3], double t, const double dir[3], double v,
                          double d, score_fn score, score_fn cross, int *jend, void *ctx)
{
  int jx = lookup(txs, tnx, pos[0], dir[0]);
  int jy = lookup(tys, tny, pos[1], dir[1]);
  int jz = lookup(tzs, tnz, pos[2], dir[2]);
  int jt = lookup(tts, tnt, t, 1.0);
  double sx = tally_s(txs, jx, pos[0], dir[0]);
  double sy = tally_s(tys, jy, pos[1], dir[1]);
  double sz = tally_s(tzs, jz, pos[2], dir[2]);
  double st = tally_st(tts, jt, t, v);
  double s_prev = 0.0;
  int64_t n = 0;
  for (;;) {
    int axis = 0; double s_min = sx;
    if (sy < s_min) { s_min = sy; axis = 1; }
    if (sz < s_min) { s_min = sz; axis = 2; }
    if (st < s_min) { s_min = st; axis = 3; }
    if (!(s_min < d)) break;
    double len = s_min - s_prev;
    if (len > 0.0) { score(ctx, jt, jz, jy, jx, len); n++; }
    if (axis == 0) { jx += (dir[0] > 0.0) ? 1 : -1; if (jx < 0 || jx >= tnx) return -1; sx = tally_s(txs, jx, pos[0], dir[0]); }
    else if (axis == 1) { jy += (dir[1] > 0.0) ? 1 : -1; if (jy < 0 || jy >= tny) return -1; sy = tally_s(tys, jy, pos[1], dir[1]); }
    else if (axis == 2) { jz += (dir[2] > 0.0) ? 1 : -1; if (jz < 0 || jz >= tnz) return -1; sz = tally_s(tzs, jz, pos[2], dir[2]); }
    else {
      if (cross) cross(ctx, jt, jz, jy, jx, 0.0);
      jt += 1; if (jt >= tnt) return -1; st = tally_st(tts, jt, t, v);
    }
    s_prev = s_min;
  }
  double len = d - s_prev;
  if (len > 0.0) { score(ctx, jt, jz, jy, jx, len); n++; }
  if (jend) { jend[0] = jt; jend[1] = jz; jend[2] = jy; jend[3] = jx; }
  return n;
}

typedef struct { int64_t *bins; double *lens; int64_t cap, n; int32_t tnx, tny, tnz; } collect_ctx;
static void collect_score(void *vc, int jt, int jz, int jy, int jx, double len)
{
  collect_ctx *c = (collect_ctx *)vc;
  if (c->n < c->cap) {
    c->bins[c->n] = (((int64_t)jt * c->tnz + jz) * c->tny + jy) * c->tnx + jx;
    c->lens[c->n] = len;
  }
  c->n++;
}
int64_t oracle_march(const double *txs, int32_t tnx, const double *tys, int32_t tny,
                     const double *tzs, int32_t tnz, const double *tts, int32_t tnt,
                     const double pos[3], double t, const double dir[3], double v,
                     double d, int64_t *bins, double *lens, int64_t cap)
{
  collect_ctx c = { bins, lens, cap, 0, tnx, tny, tnz };
  return march_core(txs, tnx, tys, tny, tzs, tnz, tts, tnt, pos, t, dir, v, d, collect_score, NULL, NULL, &c);
}

/* C.8 uniform-weight comb tooth positions */
void oracle_comb_indices(uint64_t N, uint64_t M, double a, uint64_t *idx)
{
  double r = (double)N / (double)M;
  for (uint64_t j = 0; j < M; ++j) {
    double pos = ((double)j + a) * r;
    uint64_t i = (uint64_t)pos; /* pos >= 0: truncation = floor */
    if (i > N - 1) i = N - 1;
    idx[j] = i;
  }
}

/* ------------------------------------------------------------------ */
/* Transport: source (C.4), flight (C.5), surface (C.6), collision      */
/* (C.7), census + comb (C.8), outputs (C.9)                            */
/* ------------------------------------------------------------------ */
enum { C_SOURCE, C_FLIGHTS, C_SEGMENTS, C_COLLISIONS, C_SCATTERS, C_CAPTURES, C_FISSIONS,
       C_SECONDARIES, C_CROSSINGS, C_REFLECTIONS, C_LEAKS, C_CENSUS, C_COMB_IN,
       C_COMB_OUT, C_LOST, C_FINGERPRINT };
enum { EV_CAPTURE = 0, EV_FISSION = 1, EV_LEAK = 2, EV_CENSUS = 3, EV_LOST = 4 };

static int bank_push(bank *b, const particle *q)
{
  if (b->n == b->cap) {
    size_t nc = b->cap ? b->cap * 2 : 1024;
    particle *nv = realloc(b->v, nc * sizeof(particle));
    if (!nv) return 0;
    b->v = nv; b->cap = nc;
  }
  b->v[b->n++] = *q;
  return 1;
}

static int sample_cdf(const double *cdf, int n, double xi)
{
  for (int j = 0; j < n; ++j) if (xi < cdf[j]) return j;
  return n - 1;
}

/* C.4 isotropic direction: mu on the x axis */
static void isotropic(double a, double b, double *ux, double *uy, double *uz)
{
  double mu = 2.0 * a - 1.0;
  double c, s; oracle_sincos2pi(b, &c, &s);
  double q = sqrt(fma(-mu, mu, 1.0));
  *ux = mu; *uy = q * c; *uz = q * s;
}

/* unit-test hook: the direction law above, as the transport loop calls it */
void oracle_isotropic(double a, double b, double *u3) { isotropic(a, b, &u3[0], &u3[1], &u3[2]); }

/* C.9 fingerprint: words r0,r1 of Philox(key=pid, counter=(ectr, 0x200+event, 0, 0)) */
static uint64_t fingerprint(uint64_t pid, uint32_t ectr, int event)
{
  draw2 d = draw(pid, ectr, (uint32_t)(B_FPRINT + event), 0);
  return ((uint64_t)d.r0 << 32) | (uint64_t)d.r1;
}

static size_t cell_of(const oracle_problem *p, const particle *q)
{
  return ((size_t)q->iz * p->ny + q->iy) * p->nx + q->ix;
}

/* C.4 source particle i of a batch */
static particle source_particle(const oracle_problem *p, uint64_t i, uint64_t seedb)
{
  particle q; memset(&q, 0, sizeof q);
  q.pid = i; q.ectr = 0; q.w = 1.0; q.t = p->src_t0;
  if (p->src_t1 > p->src_t0) {         /* C.17 */
    draw2 dt = draw(q.pid, 0, B_SRC_TIME, seedb);
    q.t = p->src_t0 + dt.a * (p->src_t1 - p->src_t0);
  }
  draw2 dxy = draw(q.pid, 0, B_SRC_XY, seedb);
  draw2 dzg = draw(q.pid, 0, B_SRC_ZG, seedb);
  if (p->src_isotropic) {
    draw2 dd = draw(q.pid, 0, B_SRC_DIR, seedb);
    isotropic(dd.a, dd.b, &q.ux, &q.uy, &q.uz);
  } else { q.ux = p->src_dir[0]; q.uy = p->src_dir[1]; q.uz = p->src_dir[2]; }
  if (p->src_kind == 0) {
    q.x = p->src_lo[0]; q.y = p->src_lo[1]; q.z = p->src_lo[2];
  } else if (p->src_kind == 1) {
    q.x = p->src_lo[0] + dxy.a * (p->src_hi[0] - p->src_lo[0]);
    q.y = p->src_lo[1] + dxy.b * (p->src_hi[1] - p->src_lo[1]);
    q.z = p->src_lo[2] + dzg.a * (p->src_hi[2] - p->src_lo[2]);
  } else if (p->src_kind == 3) {
    /* C.18: uniform in the ball of centre src_lo and radius src_hi[0]: the radius is R max(xi1, xi2, xi3)
     * (its distribution function is r^3), the direction from the centre is isotropic (the SRC_PIN block) */
    draw2 dp = draw(q.pid, 0, B_SRC_PIN, seedb);
    double m = dxy.a; if (dxy.b > m) m = dxy.b; if (dzg.a > m) m = dzg.a;
    const double r = p->src_hi[0] * m;
    double wx, wy, wz; isotropic(dp.a, dp.b, &wx, &wy, &wz);
    q.x = p->src_lo[0] + r * wx; q.y = p->src_lo[1] + r * wy; q.z = p->src_lo[2] + r * wz;
  } else {
    draw2 dp = draw(q.pid, 0, B_SRC_PIN, seedb);
    int64_t pin = (int64_t)(dp.a * (double)p->n_pins);
    if (pin > p->n_pins - 1) pin = p->n_pins - 1;
    int32_t c = p->pin_cell[pin];
    int ix = c % p->nx, iy = (c / p->nx) % p->ny;
    double cx = 0.5 * (p->xs[ix] + p->xs[ix + 1]), cy = 0.5 * (p->ys[iy] + p->ys[iy + 1]);
    double rho = p->radius[c] * sqrt(dp.b);
    double cc, ss; oracle_sincos2pi(dxy.a, &cc, &ss);
    q.x = cx + rho * cc; q.y = cy + rho * ss;
    q.z = p->src_lo[2] + dzg.a * (p->src_hi[2] - p->src_lo[2]);
  }
  q.g = sample_cdf(p->cdf_src, p->G, dzg.b);
  q.ix = lookup(p->xs, p->nx, q.x, q.ux);
  q.iy = lookup(p->ys, p->ny, q.y, q.uy);
  q.iz = lookup(p->zs, p->nz, q.z, q.uz);
  size_t c = cell_of(p, &q);
  q.inside = 0;
  if (p->mat_inner[c] >= 0) {
    double cx = 0.5 * (p->xs[q.ix] + p->xs[q.ix + 1]), cy = 0.5 * (p->ys[q.iy] + p->ys[q.iy + 1]);
    double dx = q.x - cx, dy = q.y - cy, R = p->radius[c];
    if (fma(dx, dx, dy * dy) < R * R) q.inside = 1;
  }
  q.reg = p->csg_n_region > 0 ? find_region(p, -1, -1, q.x, q.y, q.z, q.t) : 0;
  return q;
}

typedef struct { oracle_problem *p; int g; double w, v; } tally_ctx;
static void tally_score(void *vc, int jt, int jz, int jy, int jx, double len)
{
  tally_ctx *c = (tally_ctx *)vc; oracle_problem *p = c->p;
  size_t idx = ((((size_t)jt * p->G + c->g) * p->tnz + jz) * p->tny + jy) * p->tnx + jx;
  /* Neumaier-compensated accumulation (C.12): the reference side carries no N*eps drift */
  double s = p->tally[idx], y = c->w * len, tsum = s + y;
  if (fabs(s) >= fabs(y)) p->tally_comp[idx] += (s - tsum) + y;
  else                    p->tally_comp[idx] += (y - tsum) + s;
  p->tally[idx] = tsum;
}

/* Time-crossing estimator (C.13): w*v into the bin of the upper time edge of time bin jt. */
static void tcross_score(void *vc, int jt, int jz, int jy, int jx, double len)
{
  (void)len;
  tally_ctx *c = (tally_ctx *)vc; oracle_problem *p = c->p;
  size_t idx = p->n_track + ((((size_t)jt * p->G + c->g) * p->tnz + jz) * p->tny + jy) * p->tnx + jx;
  double s = p->tally[idx], y = c->w * c->v, tsum = s + y;
  if (fabs(s) >= fabs(y)) p->tally_comp[idx] += (s - tsum) + y;
  else                    p->tally_comp[idx] += (y - tsum) + s;
  p->tally[idx] = tsum;
}

/* Follows q0 and, depth-first, all its descendants until each is dead or
 * censused at t_k.  cnt = this (batch, step) counter row.  Returns 0 ok, 2 no memory. */
static int run_particle(oracle_problem *p, particle q0, uint64_t seedb, double t_k,
                        int last_step, bank *stack, bank *census, uint64_t *cnt)
{
  const int G = p->G;
  /* time bin whose upper edge is the census time of this step (-1: time-independent run) */
  int k_edge = -1;
  for (int j = 0; j < p->tnt; ++j) if (p->tts[j + 1] == t_k) k_edge = j;
  stack->n = 0;
  if (!bank_push(stack, &q0)) return 2;
  while (stack->n > 0) {
    particle q = stack->v[--stack->n];
    int alive = 1;
    while (alive) {
      /* C.1: the flight counter is a 24-bit field of the random-number counter; a particle that reaches
       * its limit (16 777 215 flights without a census or a new id) would repeat its streams: it ends as
       * lost, with a flight of length 0, and the run is invalid */
      if (q.ectr == 0xFFFFFFu) {
        cnt[C_LOST] += 1; cnt[C_FLIGHTS] += 1;
        cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_LOST);
        break;
      }
      const int csg = p->csg_n_region > 0;
      if (csg && q.reg < 0) {             /* C.18: born (or arrived) where no region is: lost */
        cnt[C_LOST] += 1; cnt[C_FLIGHTS] += 1;
        cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_LOST);
        break;
      }
      size_t c = cell_of(p, &q);
      int m = csg ? p->csg_rmat[q.reg] : (q.inside ? p->mat_inner[c] : p->mat_outer[c]);
      double st = p->sigma_t[m * G + q.g], v = p->speed[q.g];
      /* step 1: distance to collision */
      draw2 dc = draw(q.pid, q.ectr, B_DCOL, seedb);
      double d_c = -oracle_log(dc.a) / st;
      if (d_c < 0.0) d_c = 0.0;
      /* step 2: distance to surface, order x, y, z, cylinder; strict < replaces */
      int surf = 0;
      double d_s = plane_distance(p->xs, q.ix, q.x, q.ux);
      double dsy = plane_distance(p->ys, q.iy, q.y, q.uy);
      if (dsy < d_s) { d_s = dsy; surf = 1; }
      double dsz = plane_distance(p->zs, q.iz, q.z, q.uz);
      if (dsz < d_s) { d_s = dsz; surf = 2; }
      if (p->mat_inner[c] >= 0) {
        double cx = 0.5 * (p->xs[q.ix] + p->xs[q.ix + 1]), cy = 0.5 * (p->ys[q.iy] + p->ys[q.iy + 1]);
        double dcy = oracle_cyl_distance(q.x, q.y, q.ux, q.uy, cx, cy, p->radius[c], q.inside);
        if (dcy < d_s) { d_s = dcy; surf = 3; }
      }
      /* C.18: the quadric surfaces of the region, in the order of its list; a moving surface (C.19) is seen from
       * its own frame: position minus its displacement at the flight's start, direction minus velocity / speed */
      double d_m = INF, tau_next = INF;
      if (csg) {
        for (int j = 0; j < 8; ++j) {
          const int e = p->csg_rsurf[q.reg * 8 + j];
          if (e == 0) break;
          const int sf = (e > 0 ? e : -e) - 1;
          double dd[3], vel[3];
          surf_motion(p, sf, q.t, dd, vel);
          const double dq = oracle_quadric_distance(p->csg_coef + (size_t)sf * 10, e > 0 ? 1.0 : -1.0,
                                                    q.x - dd[0], q.y - dd[1], q.z - dd[2],
                                                    q.ux - vel[0] / v, q.uy - vel[1] / v, q.uz - vel[2] / v);
          if (dq < d_s) { d_s = dq; surf = 4 + j; }
        }
        /* C.19: the flight stops at the next break time of the surfaces' motion */
        for (int j = p->mv_n_tau - 1; j >= 0; --j) if (p->mv_tau[j] > q.t) tau_next = p->mv_tau[j];
        if (tau_next < INF) { d_m = (tau_next - q.t) * v; if (d_m < 0.0) d_m = 0.0; }
      }
      /* step 3: distance to census */
      double d_t = (t_k - q.t) * v;
      if (d_t < 0.0) d_t = 0.0;
      /* step 4: event select, ties to the earlier entry */
      double d = d_c; int ev = 0;
      if (d_s < d) { d = d_s; ev = 1; }
      if (d_t < d) { d = d_t; ev = 2; }
      if (d_m < d) { d = d_m; ev = 3; }
      /* C.16: a delayed neutron whose emission time lies at or beyond the census time waits (as its
       * precursor) in the census bank: census event of length 0, no score, its time is kept */
      const int waiting = q.t >= t_k;
      if (waiting) { d = 0.0; ev = 2; }
      /* step 5: tally march (never creates events, never draws) */
      double pos[3] = { q.x, q.y, q.z }, dir[3] = { q.ux, q.uy, q.uz };
      tally_ctx tc = { p, q.g, q.w, v };
      int jend[4];
      /* (C.14: an inactive cycle of the eigenvalue mode scores nothing and counts no segments) */
      int64_t ns = (!p->cur_score || waiting) ? 0 :
                   march_core(p->txs, p->tnx, p->tys, p->tny, p->tzs, p->tnz, p->tts, p->tnt,
                              pos, q.t, dir, v, d, tally_score, p->time_crossing ? tcross_score : NULL,
                              jend, &tc);
      if (ns < 0) { /* left the tally mesh: cannot happen when the mesh covers the domain */
        cnt[C_LOST] += 1; cnt[C_FLIGHTS] += 1;
        cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_LOST);
        break;
      }
      cnt[C_SEGMENTS] += (uint64_t)ns;
      /* step 6: move, snap */
      q.x = fma(d, q.ux, q.x); q.y = fma(d, q.uy, q.y); q.z = fma(d, q.uz, q.z);
      q.t = q.t + d / v;
      /* step 7: dispatch */
      if (ev == 2) {                       /* C.8 census */
        /* the particle is alive at the census time, which is a tally time edge (C.13) */
        if (p->time_crossing && k_edge >= 0 && !waiting) tcross_score(&tc, k_edge, jend[1], jend[2], jend[3], 0.0);
        if (!waiting) q.t = t_k;
        cnt[C_CENSUS] += 1;
        cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_CENSUS);
        cnt[C_FLIGHTS] += 1; q.ectr += 1;
        if (!last_step && !bank_push(census, &q)) return 2;
        break;
      } else if (ev == 3) {                /* C.19 break time of the surfaces' motion: nothing else happens */
        q.t = tau_next; cnt[C_CROSSINGS] += 1;
      } else if (ev == 1 && surf >= 4) {   /* C.18 quadric surface: the region on its other side */
        const int e = p->csg_rsurf[q.reg * 8 + (surf - 4)];
        q.reg = find_region(p, q.reg, (e > 0 ? e : -e) - 1, q.x, q.y, q.z, q.t);
        cnt[C_CROSSINGS] += 1;
      } else if (ev == 1) {                /* C.6 surface */
        if (surf == 3) { q.inside ^= 1; cnt[C_CROSSINGS] += 1; }
        else {
          const double *pl = surf == 0 ? p->xs : surf == 1 ? p->ys : p->zs;
          int n = surf == 0 ? p->nx : surf == 1 ? p->ny : p->nz;
          int32_t *idx = surf == 0 ? &q.ix : surf == 1 ? &q.iy : &q.iz;
          double *co = surf == 0 ? &q.x : surf == 1 ? &q.y : &q.z;
          double *u = surf == 0 ? &q.ux : surf == 1 ? &q.uy : &q.uz;
          int up = *u > 0.0;
          *co = up ? pl[*idx + 1] : pl[*idx];
          int outer = up ? (*idx == n - 1) : (*idx == 0);
          if (!outer) { *idx += up ? 1 : -1; q.inside = 0; cnt[C_CROSSINGS] += 1; }
          else if (p->bc[2 * surf + up] == 1) { *u = -*u; cnt[C_REFLECTIONS] += 1; }
          else {
            cnt[C_LEAKS] += 1; cnt[C_FLIGHTS] += 1;
            cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_LEAK);
            break;
          }
        }
      } else {                             /* C.7 collision */
        cnt[C_COLLISIONS] += 1;
        draw2 dr = draw(q.pid, q.ectr, B_REACT, seedb);
        double a = dr.a * st;
        double ssr = p->sigma_s_row[m * G + q.g];
        int ic_scatter = 0;
        if (p->ic_on) {
          /* C.15 implicit capture: the capture is taken out of the weight, the reaction is chosen among
           * scattering and fission; then the weight roulette */
          const double sf = p->sigma_f[m * G + q.g];
          const double surv = ssr + sf;
          int killed = !(surv > 0.0);
          if (!killed) {
            q.w = q.w * (surv / st);
            if (q.w < p->ic_w_roulette) {
              draw2 rr = draw(q.pid, q.ectr, B_ROULETTE, seedb);
              if (rr.a * p->ic_w_survive < q.w) q.w = p->ic_w_survive; else killed = 1;
            }
          }
          if (killed) {
            cnt[C_CAPTURES] += 1; cnt[C_FLIGHTS] += 1;
            cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_CAPTURE);
            break;
          }
          a = dr.a * surv;
          ic_scatter = !(sf > 0.0);          /* (a rounded up to surv must not turn into a fission) */
        }
        if (a < ssr || ic_scatter) {
          q.g = sample_cdf(p->cdf_s + ((size_t)m * G + q.g) * G, G, dr.b);
          draw2 dd = draw(q.pid, q.ectr, B_SCAT_DIR, seedb);
          isotropic(dd.a, dd.b, &q.ux, &q.uy, &q.uz);
          cnt[C_SCATTERS] += 1;
        } else if (a < ssr + p->sigma_f[m * G + q.g]) {
          draw2 dn = draw(q.pid, q.ectr, B_FIS_N, seedb);
          /* C.14: in a generation of the eigenvalue mode the yield is normalised by the running k */
          double yield = p->cur_k > 0.0 ? p->nu[m * G + q.g] / p->cur_k : p->nu[m * G + q.g];
          int n = (int)(yield + dn.a); /* >= 0: truncation = floor */
          for (int j = 0; j < n; ++j) {
            particle ch = q;
            draw2 di = draw(q.pid, q.ectr, (uint32_t)(B_CHILD + j), seedb);
            ch.pid = (1ull << 63) | ((((uint64_t)di.r0 << 32) | (uint64_t)di.r1) >> 1);
            ch.ectr = 0;
            draw2 cg = draw(ch.pid, 0, B_SRC_ZG, seedb);
            const double *cdf_g = p->cdf_chi + m * G;
            if (p->dn_J > 0) {
              /* C.16: prompt with probability nu_p / nu, else delayed from precursor group j with
               * probability nu_d,j / nu: emitted after an exponential delay, with the group's spectrum */
              const int J = p->dn_J;
              const double a_t = cg.a * p->nu[m * G + q.g];
              double run = p->dn_nu_prompt[m * G + q.g];
              if (!(a_t < run)) {
                int jd = J - 1;
                for (int jj = 0; jj < J; ++jj) {
                  run = run + p->dn_nu[((size_t)m * G + q.g) * J + jj];
                  if (a_t < run) { jd = jj; break; }
                }
                draw2 de = draw(ch.pid, 0, B_DELAY, seedb);
                ch.t = q.t + (-oracle_log(de.a)) / p->dn_lambda[m * J + jd];
                cdf_g = p->dn_cdf_chi + ((size_t)m * J + jd) * G;
              }
            }
            ch.g = sample_cdf(cdf_g, G, cg.b);
            draw2 cd = draw(ch.pid, 0, B_SRC_DIR, seedb);
            isotropic(cd.a, cd.b, &ch.ux, &ch.uy, &ch.uz);
            if (p->cur_k > 0.0) {
              /* C.14: the child is banked for the next generation, not followed */
              cnt[C_CENSUS] += 1;
              cnt[C_FINGERPRINT] += fingerprint(ch.pid, 0, EV_CENSUS);
              if (!last_step && !bank_push(census, &ch)) return 2;
            } else if (!bank_push(stack, &ch)) return 2;
          }
          cnt[C_FISSIONS] += 1; cnt[C_SECONDARIES] += (uint64_t)n; cnt[C_FLIGHTS] += 1;
          cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_FISSION);
          break;
        } else {
          cnt[C_CAPTURES] += 1; cnt[C_FLIGHTS] += 1;
          cnt[C_FINGERPRINT] += fingerprint(q.pid, q.ectr, EV_CAPTURE);
          break;
        }
      }
      cnt[C_FLIGHTS] += 1; q.ectr += 1;
    }
  }
  return 0;
}

/* C.8 canonical order: pid ascending; ties by the bit patterns of (t,x,y,z) */
static uint64_t bits_of(double x) { uint64_t b; memcpy(&b, &x, 8); return b; }
static int cmp_particle(const void *va, const void *vb)
{
  const particle *a = (const particle *)va, *b = (const particle *)vb;
  if (a->pid != b->pid) return a->pid < b->pid ? -1 : 1;
  uint64_t ka[4] = { bits_of(a->t), bits_of(a->x), bits_of(a->y), bits_of(a->z) };
  uint64_t kb[4] = { bits_of(b->t), bits_of(b->x), bits_of(b->y), bits_of(b->z) };
  for (int i = 0; i < 4; ++i) if (ka[i] != kb[i]) return ka[i] < kb[i] ? -1 : 1;
  return 0;
}

int oracle_run(oracle_problem *p, uint64_t seed, uint64_t n_hist, uint32_t n_batch)
{
  if (!p || n_batch == 0) return 1;
  if (p->src_kind == 3 && p->csg_n_region == 0) return 1;
  const uint32_t K = p->n_steps;
  free(p->counters);
  p->counters = calloc((size_t)n_batch * K * ORACLE_N_COUNTERS, sizeof(uint64_t));
  const int eig = p->eig_active > 0;
  free(p->k_cycle); p->k_cycle = NULL;
  if (eig) p->k_cycle = calloc((size_t)n_batch * K, sizeof(double));
  memset(p->sum1, 0, p->n_tally * sizeof(double));
  memset(p->sum2, 0, p->n_tally * sizeof(double));
  p->n_batch_done = 0; p->n_hist_per_batch = n_hist;
  bank active = { 0, 0, 0 }, census = { 0, 0, 0 }, stack = { 0, 0, 0 };
  int rc = 0;
  for (uint32_t b = 0; b < n_batch && rc == 0; ++b) {
    const uint64_t seedb = seed + (uint64_t)b;
    memset(p->tally, 0, p->n_tally * sizeof(double));
    memset(p->tally_comp, 0, p->n_tally * sizeof(double));
    active.n = 0;
    uint64_t *cnt0 = p->counters + (size_t)b * K * ORACLE_N_COUNTERS;
    for (uint64_t i = 0; i < n_hist; ++i) {
      particle q = source_particle(p, i, seedb);
      if (!bank_push(&active, &q)) { rc = 2; break; }
    }
    cnt0[C_SOURCE] += n_hist;
    double k_run = eig ? p->eig_k0 : 0.0;
    for (uint32_t k = 0; k < K && rc == 0; ++k) {
      p->cur_k = k_run;
      p->cur_score = !eig || (int32_t)k >= p->eig_inactive;
      uint64_t *cnt = cnt0 + (size_t)k * ORACLE_N_COUNTERS;
      const double t_k = p->n_census > 0 ? p->t_census[k] : INF;
      const int last = (k == K - 1);
      census.n = 0;
      for (size_t i = 0; i < active.n && rc == 0; ++i)
        rc = run_particle(p, active.v[i], seedb, t_k, last, &stack, &census, cnt);
      if (eig && rc == 0) {
        /* C.14: generation estimate of cycle k; it normalises the next cycle.  In the last cycle the
         * children are counted (census counter), not banked */
        const uint64_t n_f = last ? cnt[C_CENSUS] : (uint64_t)census.n;
        k_run = k_run * (double)n_f / (double)n_hist;
        p->k_cycle[(size_t)b * K + k] = k_run;
        if (n_f == 0) { rc = 1; break; }   /* the population died out: no next generation */
      }
      if (rc || last) break;
      if (p->comb_target > 0 || eig) {
        const uint64_t M = eig ? n_hist : p->comb_target, N = census.n;
        qsort(census.v, census.n, sizeof(particle), cmp_particle);
        cnt[C_COMB_IN] += N;
        active.n = 0;
        if (N == 0) continue;
        if (p->ic_on) {
          /* C.15 weighted comb on fixed-point weights q_i = floor(w_i 2^32 + 1/2): integer prefix sums
           * are exact, so the teeth do not depend on the order of summation */
          uint64_t *pre = malloc((N + 1) * sizeof(uint64_t));
          if (!pre) { rc = 2; break; }
          pre[0] = 0;
          for (uint64_t i = 0; i < N && rc == 0; ++i) {
            const double w = census.v[i].w;
            if (!(w >= 0.0) || !(w < 524288.0)) { rc = 1; break; }
            pre[i + 1] = pre[i] + (uint64_t)(w * 4294967296.0 + 0.5);
            if (pre[i + 1] >> 63) rc = 1;
          }
          const uint64_t Wq = pre[N];
          if (rc == 0 && Wq > 0) {
            uint32_t key[2] = { 0xFFFFFFFFu, 0xFFFFFFFFu };
            uint32_t ctr[4] = { k + 1, 0, (uint32_t)seedb, (uint32_t)(seedb >> 32) }, o[4];
            oracle_philox4x32_10(key, ctr, o);
            const double a = oracle_uniform52(o[0], o[1]);
            const double r = (double)Wq / (double)M;
            const double w_out = ((double)Wq * (1.0 / 4294967296.0)) / (double)M;
            for (uint64_t j = 0; j < M; ++j) {
              double pos = ((double)j + a) * r;
              uint64_t t = (uint64_t)pos;
              if (t > Wq - 1) t = Wq - 1;
              /* the largest i with pre[i] <= t (binary search; entries of weight 0 are never taken) */
              uint64_t lo = 0, hi = N;   /* invariant: pre[lo] <= t < pre[hi] */
              while (hi - lo > 1) { uint64_t mid = lo + (hi - lo) / 2; if (pre[mid] <= t) lo = mid; else hi = mid; }
              particle s = census.v[lo];
              s.w = w_out;
              s.pid = (1ull << 62) | ((uint64_t)(k + 1) << 40) | j;
              s.ectr = 0;
              if (!bank_push(&active, &s)) { rc = 2; break; }
            }
            cnt[C_COMB_OUT] += M;
          }
          free(pre);
          continue;
        }
        for (size_t i = 1; i < census.n; ++i)
          if (census.v[i].w != census.v[0].w) { rc = 1; break; } /* uniform-weight comb only */
        uint32_t key[2] = { 0xFFFFFFFFu, 0xFFFFFFFFu };
        uint32_t ctr[4] = { k + 1, 0, (uint32_t)seedb, (uint32_t)(seedb >> 32) }, o[4];
        oracle_philox4x32_10(key, ctr, o);
        const double a = oracle_uniform52(o[0], o[1]);
        const double r = (double)N / (double)M;
        for (uint64_t j = 0; j < M; ++j) {
          double pos = ((double)j + a) * r;
          uint64_t idx = (uint64_t)pos;
          if (idx > N - 1) idx = N - 1;
          particle s = census.v[idx];
          s.w = eig ? 1.0 : s.w * r;       /* C.14: a generation starts with unit weights */
          s.pid = (1ull << 62) | ((uint64_t)(k + 1) << 40) | j;
          s.ectr = 0;
          if (!bank_push(&active, &s)) { rc = 2; break; }
        }
        cnt[C_COMB_OUT] += M;
      } else {
        bank tmp = active; active = census; census = tmp;
      }
    }
    /* batch close-out (A14): x_b = sum + compensation; Sum x, Sum x^2 */
    for (size_t i = 0; i < p->n_tally; ++i) {
      double xb = p->tally[i] + p->tally_comp[i];
      p->tally[i] = xb;
      p->sum1[i] += xb; p->sum2[i] += xb * xb;
    }
    p->n_batch_done = b + 1;
  }
  free(active.v); free(census.v); free(stack.v);
  if (rc == 2) return 2;
  if (rc == 1) return 1;
  for (uint32_t b = 0; b < n_batch; ++b)
    for (uint32_t k = 0; k < K; ++k)
      if (p->counters[((size_t)b * K + k) * ORACLE_N_COUNTERS + C_LOST]) return 6;
  return 0;
}

/* C.14 eigenvalue mode: n_inactive + n_active generations of n_hist_per_batch particles each */
int oracle_set_eigenvalue(oracle_problem *p, int32_t n_inactive, int32_t n_active, double k0)
{
  if (!p || n_inactive < 0 || n_active < 1 || !(k0 > 0.0) || p->n_census != 0 || p->time_crossing || p->ic_on) return 1;
  p->eig_inactive = n_inactive; p->eig_active = n_active; p->eig_k0 = k0;
  p->n_steps = (uint32_t)(n_inactive + n_active);
  return 0;
}

int oracle_keff_read(const oracle_problem *p, uint32_t batch, double *k_cycle, size_t n)
{
  if (!p || !p->k_cycle || !k_cycle || batch >= p->n_batch_done || n != p->n_steps) return 1;
  memcpy(k_cycle, p->k_cycle + (size_t)batch * p->n_steps, n * sizeof(double));
  return 0;
}

/* C.18 quadric-surface CSG inside the one lattice cell */
int oracle_set_csg(oracle_problem *p, int32_t n_surf, const double *coef, int32_t n_region,
                   const int32_t *region_surf, const int32_t *region_mat)
{
  if (!p || !coef || !region_surf || !region_mat || p->csg_n_region) return 1;
  if (n_surf < 1 || n_surf > 32 || n_region < 1 || n_region > 256) return 1;
  if (p->nx != 1 || p->ny != 1 || p->nz != 1 || p->mat_inner[0] >= 0) return 1;
  for (int q = 0; q < n_region; ++q) {
    if (region_mat[q] < 0 || region_mat[q] >= p->M) return 1;
    if (region_surf[q * 8] == 0) return 1;
    for (int j = 0; j < 8; ++j) {
      const int e = region_surf[q * 8 + j];
      if (e == 0) { for (int i = j; i < 8; ++i) if (region_surf[q * 8 + i] != 0) return 1; break; }
      if ((e > 0 ? e : -e) > n_surf) return 1;
    }
  }
  for (int i = 0; i < n_surf * 10; ++i) if (!(coef[i] == coef[i]) || coef[i] == INF || coef[i] == -INF) return 1;
  p->csg_coef = dup_mem(coef, sizeof(double) * n_surf * 10);
  p->csg_rsurf = dup_mem(region_surf, sizeof(int32_t) * n_region * 8);
  p->csg_rmat = dup_mem(region_mat, sizeof(int32_t) * n_region);
  p->csg_n_surf = n_surf; p->csg_n_region = n_region;
  return 0;
}

/* C.19 moving surfaces: velocities of the intervals by one divide per component */
int oracle_set_surface_motion(oracle_problem *p, int32_t n_tau, const double *tau, const double *disp)
{
  if (!p || !tau || !disp || p->csg_n_surf == 0 || p->mv_n_tau || n_tau < 2 || n_tau > 32) return 1;
  if (!ascending(tau, n_tau)) return 1;
  const int S = p->csg_n_surf;
  for (int i = 0; i < S * n_tau * 3; ++i) if (!(disp[i] == disp[i]) || disp[i] == INF || disp[i] == -INF) return 1;
  for (int j = 0; j < n_tau; ++j) if (!(tau[j] > -INF) || !(tau[j] < INF)) return 1;
  p->mv_tau = dup_mem(tau, sizeof(double) * n_tau);
  p->mv_disp = dup_mem(disp, sizeof(double) * S * n_tau * 3);
  p->mv_vel = calloc((size_t)S * n_tau * 3, sizeof(double));
  for (int s = 0; s < S; ++s)
    for (int k = 0; k + 1 < n_tau; ++k)
      for (int i = 0; i < 3; ++i)
        p->mv_vel[((size_t)s * n_tau + k) * 3 + i] =
            (disp[((size_t)s * n_tau + k + 1) * 3 + i] - disp[((size_t)s * n_tau + k) * 3 + i]) / (tau[k + 1] - tau[k]);
  p->mv_n_tau = n_tau;
  return 0;
}

/* C.17: the source emits uniformly in time over [t0, t_end] (t0 of oracle_create); a source particle born
 * at or beyond a census time waits in the census bank like a precursor (C.16) */
int oracle_set_source_window(oracle_problem *p, double t_end)
{
  if (!p || !(t_end > p->src_t0) || !(t_end < INF)) return 1;
  p->src_t1 = t_end;
  return 0;
}

/* C.16 delayed neutrons: J precursor groups; nu_delayed [n_mat][G][J], decay [n_mat][J] (> 0),
 * chi_delayed [n_mat][J][G] (rows of a fissile material sum to 1).  nu of oracle_create stays the TOTAL
 * yield: sum_j nu_delayed <= nu required.  0 ok, 1 invalid. */
int oracle_set_delayed(oracle_problem *p, int32_t J, const double *nu_delayed, const double *decay,
                       const double *chi_delayed)
{
  if (!p || J < 1 || J > 8 || !nu_delayed || !decay || !chi_delayed || p->dn_J) return 1;
  const int M = p->M, G = p->G;
  double *nud = dup_mem(nu_delayed, sizeof(double) * M * G * J), *lam = dup_mem(decay, sizeof(double) * M * J);
  double *nup = calloc((size_t)M * G, sizeof(double)), *cdf = calloc((size_t)M * J * G, sizeof(double));
  int bad = !nud || !lam || !nup || !cdf;
  for (int m = 0; m < M && !bad; ++m) {
    int fissile = 0;
    for (int g = 0; g < G; ++g) {
      double sd = 0.0;
      for (int j = 0; j < J; ++j) { const double x = nud[((size_t)m * G + g) * J + j]; if (!(x >= 0.0)) bad = 1; sd = sd + x; }
      if (sd > p->nu[m * G + g]) bad = 1;
      nup[m * G + g] = p->nu[m * G + g] - sd;
      if (p->sigma_f[m * G + g] > 0.0) fissile = 1;
    }
    for (int j = 0; j < J; ++j) {
      if (!(lam[m * J + j] > 0.0)) bad = 1;
      const double *row = chi_delayed + ((size_t)m * J + j) * G;
      double tot = 0.0;
      for (int g = 0; g < G; ++g) { if (!(row[g] >= 0.0)) bad = 1; tot = tot + row[g]; }
      if (fissile && fabs(tot - 1.0) > 1e-12) bad = 1;
      make_cdf(row, G, tot, cdf + ((size_t)m * J + j) * G);
    }
  }
  if (bad) { free(nud); free(lam); free(nup); free(cdf); return 1; }
  p->dn_J = J; p->dn_nu = nud; p->dn_nu_prompt = nup; p->dn_lambda = lam; p->dn_cdf_chi = cdf;
  return 0;
}

/* C.15: w_roulette = 0 switches the roulette off; else 0 < w_roulette <= w_survive */
int oracle_set_implicit_capture(oracle_problem *p, double w_roulette, double w_survive)
{
  if (!p || p->eig_active > 0 || !(w_roulette >= 0.0) || (w_roulette > 0.0 && !(w_survive >= w_roulette)) ||
      !(w_survive < 524288.0)) return 1;
  p->ic_on = 1; p->ic_w_roulette = w_roulette; p->ic_w_survive = w_survive;
  return 0;
}

/* C.15 weighted comb of N weights to M teeth (unit-test hook; the same statements as in oracle_run) */
int oracle_comb_weighted(uint64_t N, uint64_t M, double a, const double *w, uint64_t *idx, double *w_out)
{
  uint64_t *pre = malloc((N + 1) * sizeof(uint64_t));
  if (!pre) return 2;
  pre[0] = 0;
  for (uint64_t i = 0; i < N; ++i) {
    if (!(w[i] >= 0.0) || !(w[i] < 524288.0)) { free(pre); return 1; }
    pre[i + 1] = pre[i] + (uint64_t)(w[i] * 4294967296.0 + 0.5);
    if (pre[i + 1] >> 63) { free(pre); return 1; }
  }
  const uint64_t Wq = pre[N];
  if (Wq == 0) { free(pre); return 1; }
  const double r = (double)Wq / (double)M;
  *w_out = ((double)Wq * (1.0 / 4294967296.0)) / (double)M;
  for (uint64_t j = 0; j < M; ++j) {
    double pos = ((double)j + a) * r;
    uint64_t t = (uint64_t)pos;
    if (t > Wq - 1) t = Wq - 1;
    uint64_t lo = 0, hi = N;
    while (hi - lo > 1) { uint64_t mid = lo + (hi - lo) / 2; if (pre[mid] <= t) lo = mid; else hi = mid; }
    idx[j] = lo;
  }
  free(pre);
  return 0;
}

size_t oracle_tally_size(const oracle_problem *p) { return p->n_tally; }
uint64_t oracle_n_steps(const oracle_problem *p) { return p->n_steps; }

int oracle_tally_read(const oracle_problem *p, int which, double *out, size_t n)
{
  if (!p || !out || n != p->n_tally || p->n_batch_done == 0) return 1;
  /* eigenvalue mode: per source particle of the active generations */
  const double B = (double)p->n_batch_done,
               N = (double)p->n_hist_per_batch * (p->eig_active > 0 ? (double)p->eig_active : 1.0);
  for (size_t i = 0; i < n; ++i) {
    if (which == 2) out[i] = p->tally[i];
    else if (which == 0) out[i] = p->sum1[i] / (B * N);
    else {
      if (p->n_batch_done < 2) { out[i] = 0.0; continue; }
      double mean = p->sum1[i] / B;
      double var = (p->sum2[i] / B - mean * mean) * (B / (B - 1.0));
      if (var < 0.0) var = 0.0;
      out[i] = sqrt(var / B) / N;
    }
  }
  return 0;
}

int oracle_counters_read(const oracle_problem *p, uint32_t batch, int32_t step, uint64_t *out16)
{
  if (!p || !p->counters || batch >= p->n_batch_done || step >= (int32_t)p->n_steps) return 1;
  memset(out16, 0, ORACLE_N_COUNTERS * sizeof(uint64_t));
  for (uint32_t k = 0; k < p->n_steps; ++k) {
    if (step >= 0 && (uint32_t)step != k) continue;
    const uint64_t *c = p->counters + ((size_t)batch * p->n_steps + k) * ORACLE_N_COUNTERS;
    for (int i = 0; i < ORACLE_N_COUNTERS; ++i) out16[i] += c[i];
  }
  return 0;
}
