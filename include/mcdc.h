/* mcdc.h — C-ABI of the B200-native event-based multigroup time-dependent
 * Monte Carlo transport path (BASELINE.json north_star: "mcdc_problem_create with
 * materials, multigroup cross sections, geometry, source, tally mesh and census
 * times; mcdc_run; mcdc_tally_read").
 *
 * What the calls compute is the per-particle history loop the paper names —
 * "transport kernels ... designed to act on a single particle" (§2),
 * fixed-source multigroup transport with time-dependent mesh tallies, time census
 * and population control (§3), track-length estimator
 * (§3.1) — run in EVENT-BASED form on one GPU (the mode PAPER.md:39
 * Fig. 1 plans and PAPER.md:55 says is not yet run).  The paper prints no
 * equations; the step-by-step definition is DESIGN.md §3.
 *
 * Conventions
 *  - Every array argument of mcdc_problem_create is a HOST pointer, caller-owned,
 *    read-only, row-major, IEEE binary64 / int32, and is copied during the call.
 *  - The library allocates only small device tables itself (cross sections, plane
 *    tables, material map: copied at create).  All large device memory — particle
 *    banks, queues, tallies, counters — lives in the caller-provided workspace
 *    (a DEVICE pointer, e.g. a torch uint8 tensor) of mcdc_workspace_bytes().
 *  - Every call returns a status; nothing throws or aborts.  mcdc_last_error()
 *    returns a thread-local description of the last failure.
 *  - There is no CPU fallback: without a CUDA device every compute call returns
 *    MCDC_ECUDA.
 */
#ifndef MCDC_H
#define MCDC_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mcdc_problem mcdc_problem; /* opaque */

typedef enum {
  MCDC_OK = 0,
  MCDC_EINVAL = 1,    /* bad argument / failed validation */
  MCDC_ENOMEM = 2,    /* workspace too small or host allocation failed */
  MCDC_ECUDA = 3,     /* CUDA runtime error or no device */
  MCDC_ESTATE = 4,    /* call out of order (e.g. read before run) */
  MCDC_EOVERFLOW = 5, /* particle bank capacity exceeded: results invalid */
  MCDC_ELOST = 6      /* a particle left the tally mesh: results invalid */
} mcdc_status;

typedef enum { MCDC_BC_VACUUM = 0, MCDC_BC_REFLECT = 1 } mcdc_bc;

/* Multigroup materials ("multigroup transport problems").
 * sigma_t,c,f, nu, chi: [n_mat][G]; sigma_s: [n_mat][G from][G to]; speed: [G] cm/s.
 * Validation: sigma_t > 0; |sigma_t - (sum_g' sigma_s + sigma_c + sigma_f)| <= 1e-12 sigma_t;
 * chi sums to 1 within 1e-12 for fissile materials.  G <= 255. */
typedef struct {
  int32_t n_mat, n_group;
  const double *sigma_t, *sigma_c, *sigma_f, *nu, *sigma_s, *chi, *speed;
} mcdc_materials;

/* Rectangular lattice of cells bounded by axis-aligned planes, each cell optionally
 * holding one z-cylinder centred in its xy cross-section (north_star item 4; the
 * restriction of PAPER.md:59 "quadric surface constructive solid geometry" that the
 * five workloads need).  xs,ys,zs: [n+1] strictly ascending, +-INFINITY allowed at
 * the ends; n <= 1023 per axis.  mat_outer, mat_inner, radius: [nz][ny][nx];
 * mat_inner = -1 means no pin; radius < half the cell's x and y widths.
 * bc: faces -x,+x,-y,+y,-z,+z. */
typedef struct {
  int32_t nx, ny, nz;
  const double *xs, *ys, *zs;
  const int32_t *mat_outer, *mat_inner;
  const double *radius;
  int32_t bc[6];
} mcdc_geometry;

/* Source at time t0, weight 1 ("fixed-source").
 * kind 0: point at lo; 1: uniform in the box [lo,hi]; 2: uniform inside the pins
 * (cells with mat_inner >= 0), z uniform in [lo[2],hi[2]]; 3 (with mcdc_set_csg): uniform in the ball of
 * centre lo and radius hi[0].
 * isotropic != 0: isotropic direction, else the unit vector dir.  group_pdf: [G]. */
typedef struct {
  int32_t kind;
  double lo[3], hi[3];
  int32_t isotropic;
  double dir[3];
  const double *group_pdf;
  double t0;
} mcdc_source;

/* Track-length tally mesh (PAPER.md:59 "time-dependent mesh tallies", :79
 * "track-length estimator"), x G groups implicit.  Plane tables [n+1] ascending;
 * must cover the geometry box; ts must contain every census time bit-for-bit.
 * Tally array index order, slowest to fastest: t, g, z, y, x. */
typedef struct {
  int32_t nx, ny, nz, nt;
  const double *xs, *ys, *zs, *ts;
  /* Time-crossing estimator ("tally ... in a logarithmically-spaced time grid with a
   * time-crossing estimator", :105; DESIGN.md §3 C.13).  When != 0 the tally array has a second block
   * of nt*G*nz*ny*nx bins behind the track-length block: bin (j, g, z, y, x) of it collects w * v_g of
   * every particle alive when the time passes the UPPER edge ts[j+1] of time bin j, in the spatial bin
   * and group it is in at that moment (a snapshot of the flux at ts[j+1]).  Runs on the pool kernel
   * only (MCDC_EINVAL when the cross-section tables do not fit in shared memory). */
  int32_t time_crossing;
} mcdc_tally_mesh;

/* Time census and population control ("time census, population control
 * techniques [9,10]").  t_census ascending, last = end time; n_census = 0 means
 * time-independent.  comb_target = 0: no combing; else the uniform-weight comb
 * brings the census bank back to comb_target particles at every census but the last. */
typedef struct {
  int32_t n_census;
  const double *t_census;
  uint64_t comb_target;
} mcdc_census;

typedef struct {
  uint64_t seed;              /* batch b uses Philox stream seed + b */
  uint64_t n_hist_per_batch;  /* source particles per batch */
  uint32_t n_batch;
  double bank_capacity_factor; /* bank slots = factor * max(n_hist_per_batch, comb_target); 0 -> 1.5 */
} mcdc_run_params;

/* Event counters, one row per (batch, census step).  Integer sums: order-independent,
 * compared exactly with the oracle.  fingerprint = wrapping sum over every terminated
 * particle of a hash of (pid, flight count, terminal event) (DESIGN.md §3 C.9). */
typedef struct {
  uint64_t source, flights, segments, collisions, scatters, captures, fissions,
      secondaries, crossings, reflections, leaks, census, comb_in, comb_out, lost,
      fingerprint;
} mcdc_counters;

/* Validates and copies the problem; builds CDF tables on the host exactly as
 * DESIGN.md §3 C.3 states and uploads them.  *out is owned by the library until
 * mcdc_problem_destroy.  MCDC_EINVAL on any validation failure. */
mcdc_status mcdc_problem_create(const mcdc_materials *mat, const mcdc_geometry *geo,
                                const mcdc_source *src, const mcdc_tally_mesh *tally,
                                const mcdc_census *census, mcdc_problem **out);

/* Bytes of device workspace mcdc_run needs for these run parameters (0 on error). */
size_t mcdc_workspace_bytes(const mcdc_problem *p, const mcdc_run_params *rp);

/* Runs n_batch batches of the whole event loop (source, flights, collisions,
 * census, comb, batch close-out) on the CUDA stream `cuda_stream` (a cudaStream_t
 * passed as void*; NULL = default stream).  workspace_dev: DEVICE pointer, 256-byte
 * aligned, at least mcdc_workspace_bytes() bytes, owned by the caller and must stay
 * alive until the last mcdc_tally_read / mcdc_counters_read.  With n_batch >= 2 two batches (eight when
 * a batch has at most 2 000 000 particles) are in flight at once (each with its own banks, queues and batch
 * tally inside the workspace; the others on library-owned streams that start after, and are joined
 * into, cuda_stream); batch b always uses Philox stream seed + b, so results do not depend on which
 * pipeline ran it.  All launches of a batch are queued without a host round trip (kernels take queue
 * lengths from a device control block); the call returns after all work is complete on the stream.
 * Calls that keep several batches in flight serialise among themselves (the streams are process-wide).
 * MCDC_EOVERFLOW / MCDC_ELOST (a particle left the tally mesh, or took 2^24 - 1 flights under one id)
 * mark the results invalid. */
mcdc_status mcdc_run(mcdc_problem *p, const mcdc_run_params *rp, void *workspace_dev,
                     size_t workspace_bytes, void *cuda_stream);

/* Number of doubles in the tally: nt * G * nz * ny * nx, twice that with the time-crossing block. */
size_t mcdc_tally_size(const mcdc_problem *p);

/* which = 0: mean per source particle over batches; 1: standard error of that mean
 * over batches (0 if n_batch < 2); 2: raw sum of w*length of the last batch.
 * out: n = mcdc_tally_size() doubles, HOST pointer if out_is_device == 0 else DEVICE
 * pointer.  Synchronises the run's stream. */
mcdc_status mcdc_tally_read(const mcdc_problem *p, int which, double *out, size_t n,
                            int out_is_device);

/* Counters of one batch; census_step = -1 sums the batch's steps. out: HOST. */
mcdc_status mcdc_counters_read(const mcdc_problem *p, uint32_t batch, int32_t census_step,
                               mcdc_counters *out);

/* k-eigenvalue mode (PAPER.md:59 "k-eigenvalue", :91 "50 inactive and 100 active cycles with 10^5
 * particles per cycle"; DESIGN.md §3 C.14).  Call after mcdc_problem_create on a time-independent
 * problem (n_census = 0, no time-crossing block) and before mcdc_workspace_bytes / mcdc_run.  Every
 * batch is then n_inactive + n_active fission generations ("steps" of mcdc_counters_read) of
 * n_hist_per_batch unit-weight particles: generation 0 is drawn from the source; a fission yields
 * floor(nu / k + xi) children, k = the running generation estimate (k0 in generation 0); children are
 * banked (they count as census events), the bank is ordered by id and combed back to n_hist_per_batch
 * particles of weight 1; k_c = k_{c-1} * (children of cycle c) / n_hist_per_batch.  Only active
 * generations score the tally; mcdc_tally_read(0, 1) are per source particle of the active
 * generations.  Runs on the pool kernel only.  MCDC_EINVAL: bad arguments, time-dependent problem, or
 * tables that do not fit in shared memory.  During mcdc_run: MCDC_EINVAL when max(nu)/k exceeds 7
 * children, MCDC_ESTATE when a generation produced no children. */
mcdc_status mcdc_set_eigenvalue(mcdc_problem *p, int32_t n_inactive, int32_t n_active, double k0);

/* Implicit capture, weight roulette and the weighted comb (PAPER.md:83 "implicit capture", :59
 * "population control techniques [9,10]"; DESIGN.md §3 C.15).  Call after mcdc_problem_create and before
 * mcdc_workspace_bytes / mcdc_run; not with the eigenvalue mode.  A collision then multiplies the weight
 * by (Sigma_s_row + Sigma_f) / Sigma_t and chooses among scattering and fission (a collision with
 * Sigma_s_row + Sigma_f = 0 ends the particle); if the new weight is below w_roulette the particle
 * survives with probability w / w_survive at weight w_survive, else it ends (both ends count as
 * captures).  w_roulette = 0: no roulette; else 0 < w_roulette <= w_survive < 2^19.  With a comb target
 * the census close is the weighted comb: weights are quantised to q = floor(w 2^32 + 1/2), tooth j sits
 * at floor((j + a) sum(q) / M) on the axis of cumulated q in id order and takes the entry whose interval
 * holds it, every survivor weighs (sum(q) 2^-32) / M.  During mcdc_run: MCDC_EINVAL when a census
 * weight is outside [0, 2^19) or the quantised total reaches 2^62.  Runs on the pool kernel only. */
mcdc_status mcdc_set_implicit_capture(mcdc_problem *p, double w_roulette, double w_survive);

/* Source with a time extent ("making the specified source active only in the first fifty
 * seconds of the simulation"; DESIGN.md §3 C.17): source particles are born uniformly in time over
 * [t0, t_end] (t0 of mcdc_source) instead of at t0.  A particle born at or beyond a census time waits in
 * the census bank until its step (as a precursor does, mcdc_set_delayed).  Call after
 * mcdc_problem_create; not with the eigenvalue mode.  Pool kernel only. */
mcdc_status mcdc_set_source_window(mcdc_problem *p, double t_end);

/* Delayed neutrons (PAPER.md:105 "delayed neutron precursor", :119 "contributions of the delayed
 * neutrons"; DESIGN.md §3 C.16).  Call after mcdc_problem_create and before mcdc_workspace_bytes /
 * mcdc_run.  J = 1..8 precursor groups; nu_delayed [n_mat][G][J] = delayed yield per fission (part of
 * the TOTAL nu given at create: their sum must not exceed it), decay [n_mat][J] > 0 (1/s), chi_delayed
 * [n_mat][J][G] (rows of a fissile material sum to 1); HOST arrays, copied.  Every fission child is then
 * prompt with probability nu_p / nu, else it comes from precursor group j with probability nu_d,j / nu:
 * its time moves on by -ln(xi) / lambda_j and its group comes from chi_delayed[j].  A particle whose
 * time is at or beyond the census time waits (as its precursor) in the census bank: one census event
 * of length 0 per census step, no score, time kept; the comb treats it like any other census particle.
 * In the eigenvalue mode the delayed data only change the spectrum of the fission source (times play no
 * part there).  Runs on the pool kernel only. */
mcdc_status mcdc_set_delayed(mcdc_problem *p, int32_t J, const double *nu_delayed, const double *decay,
                             const double *chi_delayed);

/* Generation estimate of k of every cycle of a batch of the last (eigenvalue) run.
 * k_cycle: HOST, n = n_inactive + n_active doubles. */
mcdc_status mcdc_keff_read(const mcdc_problem *p, uint32_t batch, double *k_cycle, size_t n);

/* Number of event-loop iterations and kernel launches of the last mcdc_run (host). */
mcdc_status mcdc_run_stats(const mcdc_problem *p, uint64_t *iterations, uint64_t *launches);

/* Which kernels the last mcdc_run used for the event loop (host): *pool = 1 when every census
 * step ran as one persistent launch of the pool kernel (particles resident in shared-memory
 * pools: the default whenever the cross-section tables fit in shared memory), 0 when it ran as
 * per-event kernels (flights | collisions) over index queues. */
mcdc_status mcdc_kernel_path(const mcdc_problem *p, int *pool);

/* Per-kernel timing of the following mcdc_run calls with CUDA events recorded on the
 * run's stream around every launch of the event kernels (measurement support for
 * the roofline figures; off by default).  kernel: 0 = the pool kernel (or, on the per-event
 * path, flights + tally), 1 = collisions of the per-event path (0 ms on the pool path).
 * ms = summed device time of those launches during the last mcdc_run. */
mcdc_status mcdc_profile(mcdc_problem *p, int enable);
mcdc_status mcdc_profile_read(const mcdc_problem *p, int kernel, double *ms, uint64_t *launches);

/* General quadric-surface constructive solid geometry ("defined on quadric surface constructive
 * solid geometry"; DESIGN.md §3 C.18).  Call after mcdc_problem_create on a problem whose lattice is ONE cell
 * without a pin: the cell's six planes stay the outer box (with their boundary conditions) and its inside is
 * divided into n_region regions, each the intersection of up to 8 half-spaces of quadric surfaces
 *   f(x,y,z) = A x^2 + B y^2 + C z^2 + D xy + E yz + F zx + G x + H y + J z + K      coef [n_surf][10], this order.
 * region_surf [n_region][8]: +(s+1): the region lies where f_s > 0; -(s+1): where f_s < 0; 0: unused (ends the
 * list).  region_mat [n_region].  HOST arrays, copied.  n_surf <= 32, n_region <= 256.  The regions must tile
 * the box: a particle that finds no region is lost (MCDC_ELOST).  A particle's side of every surface of its
 * region is logical (never re-derived from its coordinates); the distance to a surface is the first root at
 * which sense * f turns negative, in the cancellation-free form.  With a CSG, source kind 3 = uniform in the
 * ball of centre lo and radius hi[0].  Pool kernel only; not with the eigenvalue mode. */
mcdc_status mcdc_set_csg(mcdc_problem *p, int32_t n_surf, const double *coef, int32_t n_region,
                         const int32_t *region_surf, const int32_t *region_mat);

/* Time-dependent surfaces (PAPER.md:59 "time-dependent surface for continuous object movement [11]", :105 "to
 * exactly model the continuous movement of the control rod banks"; DESIGN.md §3 C.19).  Call after mcdc_set_csg:
 * surface s is translated by d_s(t), piecewise linear in time through disp [n_surf][n_tau][3] at the break
 * times tau [n_tau] (strictly ascending, 2 <= n_tau <= 32), constant before the first and after the last.
 * A flight sees a moving surface from the surface's frame (position minus displacement, direction minus
 * velocity / speed) and stops at every break time (a zero-effect event counted as a crossing). */
mcdc_status mcdc_set_surface_motion(mcdc_problem *p, int32_t n_tau, const double *tau, const double *disp);

/* Multi-GPU replicas (PAPER.md:55 "MPI4Py", :97-99 scaling).  The path shards by batch
 * with no exchange step: every rank runs its own batches (seed offsets chosen by the caller, batch b of a
 * rank uses seed + b) and holds a full tally replica.  After mcdc_run, the replicas are combined by ONE
 * sum all-reduce of the running sums and one of the counters, issued by the caller (NCCL through
 * torch.distributed, on the run's stream, in place on the workspace):
 *   mcdc_replica_layout: byte offsets into the workspace of sum x [n_tally doubles], sum x^2 [n_tally
 *     doubles; it sits behind sum x, 256-byte aligned, so one collective over the span
 *     [sum1_offset, sum2_offset + 8 n_tally) covers both] and of the counters
 *     [n_batch][n_steps][16] uint64 (wrapping sums: a 64-bit integer sum all-reduce is exact);
 *   mcdc_replica_commit: call after the collectives; n_ranks = number of replicas summed.  From then on
 *     mcdc_tally_read(0 | 1) returns the mean and the standard error over all n_batch * n_ranks batches and
 *     mcdc_counters_read(b, k) the sum over the ranks' batches b.  Synchronises the run's stream. */
mcdc_status mcdc_replica_layout(const mcdc_problem *p, size_t *sum1_offset, size_t *sum2_offset,
                                size_t *counters_offset, size_t *counters_bytes);
mcdc_status mcdc_replica_commit(mcdc_problem *p, uint32_t n_ranks);

/* Batch statistics for callers that must not allocate device memory (code under CUDA graph capture, serving
 * loops): the batch close-out of mcdc_run ("time-dependent mesh tallies"; SURVEY section 8(a) row A14,
 * DESIGN.md section 3 C.9) and the mean / standard error of mcdc_tally_read(0 | 1) in one call that needs no problem
 * handle and no workspace.  batches_dev: DEVICE, [n_batch][n] raw batch tallies (what mcdc_tally_read(which = 2)
 * returns for one batch), read in batch order; mean_dev, stderr_dev: DEVICE, n doubles each, caller-owned
 * (stderr_dev may be NULL; it is 0 when n_batch < 2); n_hist_per_batch: source particles per batch (times the
 * active cycles in the eigenvalue mode).  Same kernels and order of operations as the workspace path, so the
 * results equal those of mcdc_run over the same batches folded in the same order, bit for bit.
 * The running sums (sum x, sum x^2) are kept in a fixed device array inside the library, 2 *
 * MCDC_NOALLOC_MAX_BINS doubles = 16 MiB on every GPU that uses the library, held until the process exits: n
 * above MCDC_NOALLOC_MAX_BINS is rejected with MCDC_EINVAL.  The call allocates nothing (no cudaMalloc / cudaFree,
 * no library routine that allocates), does not synchronise: the launches are queued on cuda_stream (a
 * cudaStream_t as void*; NULL = default stream) and the outputs are complete when the stream reaches them.  The
 * first call on a device looks up the array's address (cudaGetSymbolAddress): make that call outside a graph
 * capture.  All calls on a device share the array: calls that overlap on the GPU race on it and must be ordered
 * by the caller (one stream, or events); nothing of an earlier call survives into a later one's results (the
 * first close-out of a call overwrites the sums). */
#define MCDC_NOALLOC_MAX_BINS ((size_t)1 << 20)
mcdc_status mcdc_batch_stats_noalloc(const double *batches_dev, uint32_t n_batch, size_t n,
                                     double n_hist_per_batch, double *mean_dev, double *stderr_dev,
                                     void *cuda_stream);

void mcdc_problem_destroy(mcdc_problem *p);
const char *mcdc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
