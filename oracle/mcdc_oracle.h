/* mcdc_oracle.h — TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded CPU oracle for the multigroup time-dependent
 * Monte Carlo history loop named by BASELINE.json `north_star` (the method of
 * PAPER.md §2-§3, lines 39, 59, 61: "transport kernels ... act on a single
 * particle on the typical history-based algorithm"; "time-dependent mesh
 * tallies, time-dependent source, time census, population control").
 * The paper prints no equations; every step follows the reading recorded in
 * DESIGN.md §3 (= SURVEY.md §8(c) C.1-C.9, App. B, App. C).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library. It shares no code, header or
 * table with the CUDA path under paper_2305_07636_b200/csrc/.
 *
 * Pins (tests/test_oracle_*.py): Philox vs torch/numpy Philox; mc_log /
 * mc_sincos2pi vs libm; closed forms S/Sigma_a, exp(-Sigma_t L), exp(alpha t),
 * e^2 = 7.389; particle balance; causality; DDA and cylinder
 * brute force; comb invariants; multigroup linear solve; eigenvalue mode: k_inf =
 * nu Sigma_f / Sigma_a, multigroup k_inf and spectrum vs numpy.linalg.eig, track-length
 * estimate of k vs the generation estimate on a leaking slab; implicit capture + roulette:
 * S/Sigma_a, (1 - e^{-Sigma_a v T})/Sigma_a and the census weight e^{-Sigma_a v T}, analog-equal
 * slab fluxes, e^{alpha t} with the weighted comb; weighted comb vs exact rational arithmetic.
 * Delayed neutrons: point-kinetics matrix exponential per census interval, 1/(Sigma_a - nu Sigma_f),
 * multigroup linear solve with delayed spectra, k_inf independent of the delayed split.
 * Parity unpinned: absolute tally values of configs 4 and 5 (no closed form).
 */
#ifndef MCDC_ORACLE_H
#define MCDC_ORACLE_H
#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One flat input record; all arrays caller-owned, copied by oracle_create. */
typedef struct {
  /* materials: [n_mat][G] except sigma_s [n_mat][G from][G to], speed [G] */
  int32_t n_mat, n_group;
  const double *sigma_t, *sigma_c, *sigma_f, *nu, *sigma_s, *chi, *speed;
  /* lattice geometry: ascending plane tables [n+1] (+-INFINITY allowed at ends) */
  int32_t nx, ny, nz;
  const double *xs, *ys, *zs;
  const int32_t *mat_outer, *mat_inner; /* [nz][ny][nx]; mat_inner -1 = no pin */
  const double *radius;                 /* [nz][ny][nx] */
  int32_t bc[6];                        /* -x,+x,-y,+y,-z,+z; 0 vacuum, 1 reflect */
  /* source */
  int32_t src_kind;                     /* 0 point, 1 box, 2 uniform in pins */
  double src_lo[3], src_hi[3];
  int32_t src_isotropic;
  double src_dir[3];
  const double *src_group_pdf;          /* [G] */
  double src_t0;
  /* tally mesh (x G implicit); index order slowest->fastest t,g,z,y,x */
  int32_t tnx, tny, tnz, tnt;
  const double *txs, *tys, *tzs, *tts;
  /* time-crossing estimator (DESIGN.md section 3 C.13): when != 0 the tally has a
   * second block of tnt*G*tnz*tny*tnx bins, one per UPPER time edge tts[j+1], scoring w*v of every
   * particle that is alive when the time passes that edge, in the spatial bin it is in */
  int32_t time_crossing;
  /* census */
  int32_t n_census;
  const double *t_census;
  uint64_t comb_target;
} oracle_input;

#define ORACLE_N_COUNTERS 16
/* order: source, flights, segments, collisions, scatters, captures, fissions,
 * secondaries, crossings, reflections, leaks, census, comb_in, comb_out, lost,
 * fingerprint */

typedef struct oracle_problem oracle_problem;

int oracle_create(const oracle_input *in, oracle_problem **out); /* 0 ok, 1 invalid */
void oracle_destroy(oracle_problem *p);
/* runs n_batch batches, seed_b = seed + b; returns 0 ok, 5 overflow, 6 lost */
int oracle_run(oracle_problem *p, uint64_t seed, uint64_t n_hist_per_batch,
               uint32_t n_batch);
/* k-eigenvalue mode (PAPER.md:59 "k-eigenvalue", :91 "50 inactive and 100 active cycles with 10^5
 * particles per cycle"; DESIGN.md section 3 C.14): call after oracle_create on a time-independent
 * problem.  Every batch is then n_inactive + n_active fission generations ("steps" of the counters)
 * of n_hist_per_batch unit-weight particles; only active generations score the tally; tally_read(0)
 * is per source particle of the active generations.  0 ok, 1 invalid. */
int oracle_set_eigenvalue(oracle_problem *p, int32_t n_inactive, int32_t n_active, double k0);
/* generation estimate of k of every cycle of a batch, n = n_inactive + n_active doubles */
int oracle_keff_read(const oracle_problem *p, uint32_t batch, double *k_cycle, size_t n);
/* Implicit capture, weight roulette and the weighted comb (PAPER.md:83 "implicit capture", :59
 * "population control techniques [9,10]"; DESIGN.md section 3 C.15).  Call after oracle_create (not with
 * the eigenvalue mode).  At a collision w *= (Sigma_s_row + Sigma_f)/Sigma_t and the reaction is chosen
 * among scattering and fission; if then w < w_roulette the particle survives with probability
 * w / w_survive at weight w_survive, else it ends (captures counter).  w_roulette = 0: no roulette.
 * The census comb becomes the weighted comb on fixed-point weights.  0 ok, 1 invalid. */
int oracle_set_implicit_capture(oracle_problem *p, double w_roulette, double w_survive);
/* Source with a time extent ("making the specified source active only in the first fifty
 * seconds of the simulation"; DESIGN.md section 3 C.17): birth time uniform in [t0, t_end].  0 ok. */
int oracle_set_source_window(oracle_problem *p, double t_end);
/* Delayed neutrons (PAPER.md:105 "delayed neutron precursor", :119 "contributions of the delayed
 * neutrons"; DESIGN.md section 3 C.16).  J precursor groups (1..8); nu_delayed [n_mat][G][J] = delayed
 * yield per fission, decay [n_mat][J] > 0, chi_delayed [n_mat][J][G].  nu of oracle_create stays the
 * TOTAL yield.  Every fission child is prompt with probability nu_p/nu, else delayed from group j with
 * probability nu_d,j/nu: emitted at t - ln(xi)/lambda_j with the group's spectrum.  A delayed neutron
 * whose emission time is at or beyond the census time waits in the census bank (census event of
 * length 0, no score, time kept).  0 ok, 1 invalid. */
int oracle_set_delayed(oracle_problem *p, int32_t J, const double *nu_delayed, const double *decay,
                       const double *chi_delayed);
/* General quadric-surface constructive solid geometry ("defined on quadric surface constructive
 * solid geometry"; DESIGN.md section 3 C.18).  Call after oracle_create on a problem whose lattice is ONE cell
 * without a pin: that cell's six planes stay the outer box (with their boundary conditions), and its inside is
 * divided into n_region regions, each the intersection of up to 8 half-spaces of quadric surfaces
 *   f(x,y,z) = A x^2 + B y^2 + C z^2 + D xy + E yz + F zx + G x + H y + J z + K   (coef [n_surf][10] in this order).
 * region_surf [n_region][8]: +(s+1) = the region lies where f_s > 0, -(s+1) = where f_s < 0, 0 = unused (the
 * list ends).  region_mat [n_region].  The regions must tile the box (a particle that finds no region is lost).
 * n_surf <= 32, n_region <= 256.  Source kind 3 becomes available: uniform in the ball of centre src_lo and
 * radius src_hi[0].  0 ok, 1 invalid. */
int oracle_set_csg(oracle_problem *p, int32_t n_surf, const double *coef, int32_t n_region,
                   const int32_t *region_surf, const int32_t *region_mat);
/* Time-dependent surfaces (PAPER.md:59 "time-dependent surface for continuous object movement [11]", :105;
 * DESIGN.md section 3 C.19): surface s is translated by d_s(t), piecewise linear in time through the
 * displacements disp [n_surf][n_tau][3] at the break times tau [n_tau] (ascending), constant before the first
 * and after the last.  A flight stops at every break time (a zero-effect event counted as a crossing).
 * n_tau <= 32.  Call after oracle_set_csg.  0 ok, 1 invalid. */
int oracle_set_surface_motion(oracle_problem *p, int32_t n_tau, const double *tau, const double *disp);
/* unit-test hook: distance along (ux,uy,uz) from (x,y,z) to the point where sense * f turns negative
 * (sense = +1 / -1: the side the particle is logically on), or +inf */
double oracle_quadric_distance(const double *coef10, double sense, double x, double y, double z,
                               double ux, double uy, double uz);
size_t oracle_tally_size(const oracle_problem *p);
/* which: 0 mean per source particle, 1 std error over batches, 2 last raw batch */
int oracle_tally_read(const oracle_problem *p, int which, double *out, size_t n);
/* census_step -1 = sum over the batch's steps */
int oracle_counters_read(const oracle_problem *p, uint32_t batch, int32_t census_step,
                         uint64_t *out16);
/* size of the census bank after each step of the last batch (pre-comb) — debug */
uint64_t oracle_n_steps(const oracle_problem *p);

/* ---- unit-test hooks: the oracle's own building blocks, exposed for pins ---- */
void oracle_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]);
double oracle_uniform52(uint32_t hi, uint32_t lo);
double oracle_log(double x);
void oracle_sincos2pi(double u, double *c, double *s);
/* C.4 isotropic direction from two uniforms: u3 = (mu, q cos phi, q sin phi) */
void oracle_isotropic(double a, double b, double *u3);
/* distance to the z-cylinder of radius R centred (cx,cy); inside=1/0 */
double oracle_cyl_distance(double x, double y, double ux, double uy, double cx,
                           double cy, double R, int inside);
/* tally march of one flight on a mesh; writes (bin index, length) pairs, returns
 * number of segments (<= cap) or -1 when the track leaves the mesh */
int64_t oracle_march(const double *txs, int32_t tnx, const double *tys, int32_t tny,
                     const double *tzs, int32_t tnz, const double *tts, int32_t tnt,
                     const double pos[3], double t, const double dir[3], double v,
                     double d, int64_t *bins, double *lens, int64_t cap);
/* uniform-weight comb indices: idx[j] = floor((j+a) N/M) clamped, j<M */
void oracle_comb_indices(uint64_t N, uint64_t M, double a, uint64_t *idx);
/* weighted comb (C.15): idx[j] = entry tooth j takes, *w_out = weight of every survivor; 0 ok */
int oracle_comb_weighted(uint64_t N, uint64_t M, double a, const double *w, uint64_t *idx, double *w_out);

#ifdef __cplusplus
}
#endif
#endif
