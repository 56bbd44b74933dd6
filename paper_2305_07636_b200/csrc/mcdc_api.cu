// mcdc_api.cu — C-ABI entry points (include/mcdc.h) and the host driver of the event
// loop: batches -> census steps -> event iterations (k_flight, k_collide, k_flip) ->
// census ordering + comb -> batch close-out.  Single translation unit: the kernel
// sources are included here so that every launch sees its kernel's definition.
#include "../../include/mcdc.h"
#include "mcdc_transport.cu"
#include "mcdc_pool.cu"
#include "mcdc_comb.cu"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <algorithm>
#include <atomic>
#include <mutex>
#include <thread>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

using namespace mcdc;

namespace {

thread_local std::string g_err;

mcdc_status fail(mcdc_status s, const char *fmt, ...)
{
  char buf[512];
  va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
  g_err = buf;
  return s;
}

#define CU(call)                                                                       \
  do {                                                                                 \
    cudaError_t e_ = (call);                                                           \
    if (e_ != cudaSuccess)                                                             \
      return fail(MCDC_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

bool ascending(const double *p, int n1)
{
  for (int i = 0; i + 1 < n1; ++i) if (!(p[i] < p[i + 1])) return false;
  return true;
}

// C.3: running sum ascending, one divide per entry, last entry exactly 1
void build_cdf(const double *pdf, int n, double total, double *cdf)
{
  double run = 0.0;
  for (int j = 0; j < n; ++j) { run = run + pdf[j]; cdf[j] = total > 0.0 ? run / total : 0.0; }
  cdf[n - 1] = 1.0;
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Layout {          // byte offsets into the caller's workspace
  // shared by all pipelines (absolute offsets)
  size_t counters, last, sum1, sum2, scratch, flag, total;
  // private to one pipeline (offsets relative to pipe_base[i])
  size_t ctl, tally, bankA, bankB, q0, q1, qcoll, qcensus, order, bcount, boffs, bcursor, tiles, wpre, wtiles, pipe_bytes;
  uint32_t n_wtiles;       // tiles of the 64-bit scan of the weighted comb
  size_t pipe_base[4];
  int n_pipe;              // batches in flight at once (2 when the run has >= 2 batches)
  uint32_t capacity, n_buckets, n_tiles;
  BucketMap bm;
};

}  // namespace

struct mcdc_problem {
  DevProblem dp{};
  TableLayout tl{};
  int use_smem = 1;
  size_t smem_bytes = 0;
  std::vector<void *> dev_allocs;
  int n_census = 0;
  std::vector<double> t_census;
  uint64_t comb_target = 0;
  uint32_t n_steps = 1;
  size_t n_tally = 0;
  int sm_count = 148, occ_move = 2, occ_collide = 2, occ_tail = 1;
  uint32_t *host_mirror = nullptr;   // pinned, mapped: n_active, n_census, overflow, bank_tail
  // state of the last run
  bool ran = false;
  void *ws = nullptr;
  Layout lay{};
  cudaStream_t stream = nullptr;
  uint32_t n_batch = 0;
  uint64_t n_hist = 0;
  std::vector<unsigned long long> counters;  // [batch][step][16]
  uint64_t iterations = 0, launches = 0;
  // optional per-kernel timing with CUDA events on the run's stream (mcdc_profile)
  // tuning knobs (env MCDC_MAX_FLIGHTS, MCDC_TAIL, MCDC_FUSE_BULK; defaults from measurement)
  int max_flights = 4;
  uint64_t tail_threshold = 148 * 256 * 2;
  int fuse_bulk = 0;
  int group = 4;                      // iterations launched per host synchronisation on very long queues
  int refill = 1;                    // persistent lanes refilled from the active queue (long queues)
  int occ_refill = 2;
  const double *vsig_dev = nullptr;  // [G] group speed x largest sigma_t of the group (comb: long histories first)
  double long_mfp = 64.0;
  int time_crossing = 0;             // the tally carries the time-crossing block (pool kernel only)
  int pool = 1;                      // one persistent pool launch per census step (mcdc_pool.cu)
  int pool_ok = 1;                   // the pool kernel can run this problem (tables fit in shared memory)
  int occ_pool = 1;
  size_t pool_smem = 0;
  // k-eigenvalue mode (mcdc_set_eigenvalue; DESIGN.md §3 C.14): both 0 = fixed source
  int eig_inactive = 0, eig_active = 0;
  double eig_k0 = 1.0, nu_max = 0.0;
  std::vector<double> host_xs4;      // host copy of (sigma_t, sigma_s_row, sigma_f, nu) per (m, g)
  int ic_on = 0;                     // implicit capture + roulette + weighted comb (mcdc_set_implicit_capture; C.15)
  std::vector<double> k_cycle;       // [batch][cycle] generation estimate of k
  int profile = 0;
  cudaEvent_t ev[48] = {};             // per pipeline: 3 per iteration of a launch group
  cudaStream_t aux_stream[3] = {nullptr, nullptr, nullptr};   // streams of pipelines 1..3
  double prof_ms[2] = {0.0, 0.0};        // k_move, k_collide
  uint64_t prof_launches[2] = {0, 0};
};

namespace {

// the instantiated variants of the pool kernel: <time-crossing, eigenvalue, implicit capture, delayed>
using PoolFn = void (*)(DevProblem, TableLayout, int, Bank, Bank, Ctl *, Queues, int, uint32_t);
const PoolFn POOL_VARIANTS[] = {
    k_pool<false, false, false, false>, k_pool<true, false, false, false>, k_pool<false, true, false, false>,
    k_pool<false, false, true, false>,  k_pool<true, false, true, false>,  k_pool<false, false, false, true>,
    k_pool<true, false, false, true>,   k_pool<false, false, true, true>,  k_pool<true, false, true, true>,
    k_pool<false, true, false, true>};
PoolFn pool_variant(bool tc, bool eig, bool ic, bool dn)
{
  if (eig) return dn ? POOL_VARIANTS[9] : POOL_VARIANTS[2];
  if (dn && ic) return tc ? POOL_VARIANTS[8] : POOL_VARIANTS[7];
  if (dn) return tc ? POOL_VARIANTS[6] : POOL_VARIANTS[5];
  if (ic) return tc ? POOL_VARIANTS[4] : POOL_VARIANTS[3];
  if (eig) return POOL_VARIANTS[2];
  return tc ? POOL_VARIANTS[1] : POOL_VARIANTS[0];
}

template <typename T>
mcdc_status upload(mcdc_problem *p, const T *host, size_t n, const T **dev)
{
  void *d = nullptr;
  CU(cudaMalloc(&d, (n ? n : 1) * sizeof(T)));
  p->dev_allocs.push_back(d);
  if (n) CU(cudaMemcpy(d, host, n * sizeof(T), cudaMemcpyHostToDevice));
  *dev = (const T *)d;
  return MCDC_OK;
}

// particles the census close combs back to: the comb target, or the generation size (C.14)
uint64_t comb_size(const mcdc_problem *p, const mcdc_run_params *rp)
{
  return p->eig_active > 0 ? rp->n_hist_per_batch : p->comb_target;
}

mcdc_status compute_layout(const mcdc_problem *p, const mcdc_run_params *rp, Layout *L)
{
  if (!rp || rp->n_batch == 0 || rp->n_hist_per_batch == 0) return fail(MCDC_EINVAL, "empty run");
  double factor = rp->bank_capacity_factor;
  if (factor == 0.0) factor = 1.5;
  if (!(factor >= 1.0)) return fail(MCDC_EINVAL, "bank_capacity_factor must be >= 1");
  const uint64_t comb_M = comb_size(p, rp);
  const uint64_t nmax = rp->n_hist_per_batch > comb_M ? rp->n_hist_per_batch : comb_M;
  const double capd = std::ceil(factor * (double)nmax) + 1024.0;
  if (capd >= 4294967295.0) return fail(MCDC_EINVAL, "bank capacity exceeds 2^32 slots");
  const uint32_t cap = (uint32_t)capd;
  L->capacity = cap;
  BucketMap &bm = L->bm;
  bm.shift_dense = 2;
  bm.nb0 = (uint32_t)((rp->n_hist_per_batch >> 2) + 1);
  bm.nb1 = (uint32_t)((comb_M >> 2) + 1);
  uint32_t bits = 1;
  while (bits < 30 && (1ull << (bits + 1)) <= (uint64_t)cap / 4) ++bits;
  bm.bits_hash = bits;
  bm.base1 = 0;
  bm.n_buckets = bm.nb0 + bm.nb1 + (1u << bits);
  L->n_buckets = bm.n_buckets;
  L->n_tiles = (bm.n_buckets + SCAN_TILE - 1) / SCAN_TILE;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align256(off + bytes); return o; };
  const bool comb = comb_M > 0 && p->n_steps > 1;
  // one pipeline's private region
  L->ctl = take(sizeof(Ctl));
  L->tally = take(p->n_tally * 8);
  L->bankA = take((size_t)cap * 80);
  L->bankB = take((size_t)cap * 80);
  L->q0 = take((size_t)cap * 4);
  L->q1 = take((size_t)cap * 4);
  L->qcoll = take((size_t)cap * 4);
  L->qcensus = take((size_t)cap * 4);
  L->order = take(comb ? (size_t)cap * 4 : 0);
  L->bcount = take(comb ? (size_t)bm.n_buckets * 4 : 0);
  L->boffs = take(comb ? (size_t)bm.n_buckets * 4 : 0);
  L->bcursor = take(comb ? (size_t)bm.n_buckets * 4 : 0);
  L->tiles = take(comb ? (size_t)L->n_tiles * 4 : 0);
  const bool wcomb = comb && p->ic_on;                 // weighted comb (C.15): fixed-point prefix sums
  L->n_wtiles = (cap + SCAN_TILE - 1) / SCAN_TILE;
  L->wpre = take(wcomb ? ((size_t)cap + 1) * 8 : 0);
  L->wtiles = take(wcomb ? (size_t)L->n_wtiles * 8 : 0);
  L->pipe_bytes = off;
  // shared region
  off = 0;
  L->counters = take((size_t)rp->n_batch * p->n_steps * N_CNT * 8);
  L->last = take(p->n_tally * 8);
  L->sum1 = take(p->n_tally * 8);
  L->sum2 = take(p->n_tally * 8);
  L->scratch = take(p->n_tally * 8);
  L->flag = take(256);
  // batches in flight (MCDC_PIPELINES = 1..4): 2; 4 when a batch cannot fill the pools by itself (a launch
  // lasts as long as its longest history, so small batches leave most warps idle: measured on the
  // eigenvalue pin cell at 1e5 particles per cycle, 2.1e8 / 3.4e8 / 4.9e8 histories/s with 1 / 2 / 4)
  int np = nmax <= 262144 ? 4 : 2;
  if (const char *e = getenv("MCDC_PIPELINES")) np = std::min(4, std::max(1, atoi(e)));
  np = (int)std::min<uint32_t>((uint32_t)np, rp->n_batch);
  L->n_pipe = np;
  for (int i = 0; i < 4; ++i) L->pipe_base[i] = off + (size_t)(i < np ? i : 0) * L->pipe_bytes;
  L->total = off + (size_t)np * L->pipe_bytes;
  return MCDC_OK;
}

Bank bank_at(char *base, size_t off, uint32_t cap)
{
  Bank B;
  char *p = base + off;
  B.xy = (double2 *)p;  p += (size_t)cap * 16;
  B.zt = (double2 *)p;  p += (size_t)cap * 16;
  B.uxy = (double2 *)p; p += (size_t)cap * 16;
  B.uzw = (double2 *)p; p += (size_t)cap * 16;
  B.idp = (ulonglong2 *)p;
  return B;
}

__global__ void k_begin_batch(Ctl *ctl, unsigned long long seedb, uint32_t n_src)
{
  ctl->n_active = n_src; ctl->n_next = 0; ctl->n_coll = 0; ctl->n_census = 0;
  ctl->bank_tail = n_src; ctl->parity = 0; ctl->overflow = 0; ctl->iter = 0;
  ctl->seedb = seedb;
}

__global__ void k_begin_step(Ctl *ctl, double t_k, uint32_t last, uint32_t k1, unsigned long long *cnt,
                             unsigned long long n_source, double eig_k, uint32_t score)
{
  ctl->eig_k = eig_k; ctl->score = score;
  ctl->t_k = t_k; ctl->last_step = last; ctl->step_k1 = k1; ctl->cnt = cnt;
  ctl->n_census = 0; ctl->n_next = 0; ctl->n_coll = 0; ctl->parity = 0; ctl->fetch = 0;
  ctl->comb_front = 0; ctl->comb_back = 0;
  if (n_source) cnt[K_SOURCE] += n_source;
}

// after a census step: either comb accounting (M > 0) or hand the census list over
__global__ void k_end_step(Ctl *ctl, unsigned long long M, uint32_t *mirror, const unsigned long long *w_pre)
{
  const uint32_t n = ctl->n_census;
  if (M) {
    ctl->cnt[K_COMB_IN] += n;
    // (weighted comb: a census bank of zero weights has no survivors)
    const bool out = n && !(w_pre && w_pre[n] == 0ull);
    if (out) ctl->cnt[K_COMB_OUT] += M;
    ctl->n_active = out ? (uint32_t)M : 0u;
    ctl->bank_tail = (uint32_t)M;
  } else { ctl->n_active = n; ctl->bank_tail = n; }
  mirror[0] = ctl->n_active; mirror[1] = n; mirror[2] = ctl->overflow; mirror[3] = ctl->bank_tail;
}

}  // namespace

extern "C" const char *mcdc_last_error(void) { return g_err.c_str(); }

extern "C" void mcdc_problem_destroy(mcdc_problem *p)
{
  if (!p) return;
  for (void *d : p->dev_allocs) cudaFree(d);
  if (p->host_mirror) cudaFreeHost(p->host_mirror);
  for (cudaEvent_t e : p->ev) if (e) cudaEventDestroy(e);
  for (cudaStream_t a : p->aux_stream) if (a) cudaStreamDestroy(a);
  delete p;
}

extern "C" mcdc_status mcdc_problem_create(const mcdc_materials *mat, const mcdc_geometry *geo,
                                           const mcdc_source *src, const mcdc_tally_mesh *tal,
                                           const mcdc_census *cen, mcdc_problem **out)
{
  if (!mat || !geo || !src || !tal || !cen || !out) return fail(MCDC_EINVAL, "null argument");
  const int M = mat->n_mat, G = mat->n_group;
  if (M < 1 || M > 127 || G < 1 || G > 255) return fail(MCDC_EINVAL, "n_mat in 1..127, n_group in 1..255");
  if (geo->nx < 1 || geo->ny < 1 || geo->nz < 1 || geo->nx > 1023 || geo->ny > 1023 || geo->nz > 1023)
    return fail(MCDC_EINVAL, "lattice size per axis must be in 1..1023");
  if (tal->nx < 1 || tal->ny < 1 || tal->nz < 1 || tal->nt < 1) return fail(MCDC_EINVAL, "empty tally mesh");
  if (!ascending(geo->xs, geo->nx + 1) || !ascending(geo->ys, geo->ny + 1) || !ascending(geo->zs, geo->nz + 1))
    return fail(MCDC_EINVAL, "lattice plane tables must be strictly ascending");
  if (!ascending(tal->xs, tal->nx + 1) || !ascending(tal->ys, tal->ny + 1) ||
      !ascending(tal->zs, tal->nz + 1) || !ascending(tal->ts, tal->nt + 1))
    return fail(MCDC_EINVAL, "tally plane tables must be strictly ascending");
  if (tal->xs[0] > geo->xs[0] || tal->xs[tal->nx] < geo->xs[geo->nx] || tal->ys[0] > geo->ys[0] ||
      tal->ys[tal->ny] < geo->ys[geo->ny] || tal->zs[0] > geo->zs[0] || tal->zs[tal->nz] < geo->zs[geo->nz])
    return fail(MCDC_EINVAL, "tally mesh does not cover the geometry box");
  if (cen->n_census < 0) return fail(MCDC_EINVAL, "n_census < 0");
  if (cen->n_census > 0 && !ascending(cen->t_census, cen->n_census))
    return fail(MCDC_EINVAL, "census times must be strictly ascending");
  for (int k = 0; k < cen->n_census; ++k) {
    bool found = false;
    for (int j = 0; j <= tal->nt; ++j) found = found || tal->ts[j] == cen->t_census[k];
    if (!found) return fail(MCDC_EINVAL, "census time %d is not a tally time edge", k);
  }
  if (tal->ts[0] > src->t0) return fail(MCDC_EINVAL, "source time before the first tally time edge");
  if (src->kind < 0 || src->kind > 2) return fail(MCDC_EINVAL, "source kind");

  // tables: [xs4 | cdf_s | cdf_chi | cdf_src | speed]  (C.3)
  TableLayout tl;
  tl.xs4 = 0; tl.cdf_s = M * G * 4; tl.cdf_chi = tl.cdf_s + M * G * G; tl.cdf_src = tl.cdf_chi + M * G;
  tl.speed = tl.cdf_src + G; tl.total = tl.speed + G;
  std::vector<double> tab(tl.total, 0.0);
  double nu_max = 0.0;
  for (int m = 0; m < M; ++m) {
    bool fissile = false;
    for (int g = 0; g < G; ++g) {
      const double *row = mat->sigma_s + ((size_t)m * G + g) * G;
      double sr = 0.0;
      for (int j = 0; j < G; ++j) { if (row[j] < 0.0) return fail(MCDC_EINVAL, "negative sigma_s"); sr = sr + row[j]; }
      const double st = mat->sigma_t[m * G + g], sc = mat->sigma_c[m * G + g], sf = mat->sigma_f[m * G + g];
      if (!(st > 0.0) || sc < 0.0 || sf < 0.0) return fail(MCDC_EINVAL, "cross sections must be >= 0, sigma_t > 0");
      if (!(mat->nu[m * G + g] >= 0.0) || mat->nu[m * G + g] > 7.0) return fail(MCDC_EINVAL, "nu must be in [0, 7]");
      if (std::fabs(st - (sr + sc + sf)) > 1e-12 * st)
        return fail(MCDC_EINVAL, "sigma_t != sigma_s_row + sigma_c + sigma_f (mat %d group %d)", m, g);
      double *x4 = &tab[tl.xs4 + (m * G + g) * 4];
      x4[0] = st; x4[1] = sr; x4[2] = sf; x4[3] = mat->nu[m * G + g];
      if (sf > 0.0 && x4[3] > nu_max) nu_max = x4[3];
      build_cdf(row, G, sr, &tab[tl.cdf_s + (m * G + g) * G]);
      fissile = fissile || sf > 0.0;
    }
    double cs = 0.0;
    for (int g = 0; g < G; ++g) cs = cs + mat->chi[m * G + g];
    if (fissile && std::fabs(cs - 1.0) > 1e-12) return fail(MCDC_EINVAL, "chi of material %d does not sum to 1", m);
    build_cdf(mat->chi + m * G, G, cs, &tab[tl.cdf_chi + m * G]);
  }
  {
    double ps = 0.0;
    for (int g = 0; g < G; ++g) ps = ps + src->group_pdf[g];
    if (std::fabs(ps - 1.0) > 1e-12) return fail(MCDC_EINVAL, "source group pdf does not sum to 1");
    build_cdf(src->group_pdf, G, ps, &tab[tl.cdf_src]);
  }
  for (int g = 0; g < G; ++g) {
    if (!(mat->speed[g] > 0.0)) return fail(MCDC_EINVAL, "group speeds must be > 0");
    tab[tl.speed + g] = mat->speed[g];
  }

  const size_t nc = (size_t)geo->nx * geo->ny * geo->nz;
  std::vector<int8_t> mo(nc), mi(nc);
  std::vector<int> pins;
  for (size_t c = 0; c < nc; ++c) {
    if (geo->mat_outer[c] < 0 || geo->mat_outer[c] >= M || geo->mat_inner[c] >= M)
      return fail(MCDC_EINVAL, "material index out of range in cell %zu", c);
    mo[c] = (int8_t)geo->mat_outer[c];
    mi[c] = (int8_t)(geo->mat_inner[c] < 0 ? -1 : geo->mat_inner[c]);
    if (geo->mat_inner[c] >= 0) {
      const int ix = (int)(c % geo->nx), iy = (int)((c / geo->nx) % geo->ny);
      const double hw = 0.5 * (geo->xs[ix + 1] - geo->xs[ix]), hh = 0.5 * (geo->ys[iy + 1] - geo->ys[iy]);
      const double R = geo->radius[c];
      if (!(R > 0.0) || !(R < hw) || !(R < hh)) return fail(MCDC_EINVAL, "pin radius of cell %zu does not fit", c);
      pins.push_back((int)c);
    }
  }
  if (src->kind == 2 && pins.empty()) return fail(MCDC_EINVAL, "pin source without pins");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(MCDC_ECUDA, "no CUDA device");

  mcdc_problem *p = new mcdc_problem();
  p->nu_max = nu_max;
  p->host_xs4.assign(tab.begin() + tl.xs4, tab.begin() + tl.xs4 + (size_t)M * G * 4);
  mcdc_status st = MCDC_OK;
  DevProblem &D = p->dp;
  D.n_mat = M; D.G = G;
  const double *dtab = nullptr;
  auto UP = [&](auto host, size_t n, auto devpp) { if (st == MCDC_OK) st = upload(p, host, n, devpp); };
  UP(tab.data(), tab.size(), &dtab);
  D.xs4 = dtab + tl.xs4; D.cdf_s = dtab + tl.cdf_s; D.cdf_chi = dtab + tl.cdf_chi;
  D.cdf_src = dtab + tl.cdf_src; D.speed = dtab + tl.speed;
  D.nx = geo->nx; D.ny = geo->ny; D.nz = geo->nz;
  UP(geo->xs, (size_t)geo->nx + 1, &D.px); UP(geo->ys, (size_t)geo->ny + 1, &D.py);
  UP(geo->zs, (size_t)geo->nz + 1, &D.pz);
  UP(mo.data(), nc, &D.mat_outer); UP(mi.data(), nc, &D.mat_inner);
  UP(geo->radius, nc, &D.radius);
  D.has_pins = pins.empty() ? 0 : 1;
  for (int i = 0; i < 6; ++i) D.bc[i] = geo->bc[i];
  D.src_kind = src->kind; D.src_isotropic = src->isotropic; D.src_t0 = src->t0; D.src_t1 = src->t0;
  for (int i = 0; i < 3; ++i) { D.src_lo[i] = src->lo[i]; D.src_hi[i] = src->hi[i]; D.src_dir[i] = src->dir[i]; }
  {
    std::vector<double> vsig(G, 0.0);
    for (int g = 0; g < G; ++g) {
      double mx = 0.0;
      for (int m = 0; m < M; ++m) mx = std::max(mx, mat->sigma_t[m * G + g]);
      vsig[g] = mat->speed[g] * mx;
    }
    UP(vsig.data(), vsig.size(), &p->vsig_dev);
  }
  D.n_pins = (long long)pins.size();
  UP(pins.data(), pins.size(), &D.pin_cell);
  D.tnx = tal->nx; D.tny = tal->ny; D.tnz = tal->nz; D.tnt = tal->nt;
  UP(tal->xs, (size_t)tal->nx + 1, &D.tx); UP(tal->ys, (size_t)tal->ny + 1, &D.ty);
  UP(tal->zs, (size_t)tal->nz + 1, &D.tz); UP(tal->ts, (size_t)tal->nt + 1, &D.tt);
  D.tally = nullptr;
  auto hint = [](const double *t, int n) {
    AxisHint h{0.0, 0.0};
    if (std::isfinite(t[0]) && std::isfinite(t[n]) && t[n] > t[0]) { h.p0 = t[0]; h.inv_w = (double)n / (t[n] - t[0]); }
    return h;
  };
  auto same = [](const double *a, int na, const double *b, int nb) {
    return na == nb && std::memcmp(a, b, sizeof(double) * (size_t)(na + 1)) == 0;
  };
  D.simple_tally = same(tal->xs, tal->nx, geo->xs, geo->nx) && same(tal->ys, tal->ny, geo->ys, geo->ny) &&
                   same(tal->zs, tal->nz, geo->zs, geo->nz);
  if (getenv("MCDC_NO_SIMPLE_TALLY")) D.simple_tally = 0;
  {
    // bins one census step / time bin keeps hot; with many more bins than lanes in flight two lanes of
    // a warp seldom meet in a bin (measured: DESIGN.md section 6)
    const size_t hot = (size_t)G * tal->nz * tal->ny * tal->nx;
    D.aggregate_tally = hot <= 4096 ? 1 : 0;
    if (const char *e = getenv("MCDC_AGG")) D.aggregate_tally = atoi(e);
  }
  D.hx = hint(tal->xs, tal->nx); D.hy = hint(tal->ys, tal->ny);
  D.hz = hint(tal->zs, tal->nz); D.ht = hint(tal->ts, tal->nt);
  if (st == MCDC_OK && cudaHostAlloc((void **)&p->host_mirror, 256, cudaHostAllocMapped) != cudaSuccess)
    st = fail(MCDC_ECUDA, "cudaHostAlloc failed");
  if (st != MCDC_OK) { mcdc_problem_destroy(p); return st; }
  p->tl = tl;
  p->smem_bytes = (size_t)tl.total * 8;
  p->use_smem = p->smem_bytes <= 40 * 1024;
  if (!p->use_smem) p->smem_bytes = 0;
  p->n_census = cen->n_census;
  p->t_census.assign(cen->t_census, cen->t_census + cen->n_census);
  p->comb_target = cen->comb_target;
  p->n_steps = cen->n_census > 0 ? (uint32_t)cen->n_census : 1u;
  p->n_tally = (size_t)tal->nt * G * tal->nz * tal->ny * tal->nx;
  D.tcross_off = -1;
  if (tal->time_crossing) { D.tcross_off = (long long)p->n_tally; p->n_tally *= 2; p->time_crossing = 1; }
  int dev = 0; cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&p->occ_move, k_flight<false, false>, BS, p->smem_bytes);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&p->occ_collide, k_collide, BS, p->smem_bytes);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&p->occ_tail, k_flight<true, true>, BS, p->smem_bytes);
  if (p->occ_tail < 1) p->occ_tail = 1;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&p->occ_refill, k_flight<false, false, true>, REFILL_THREADS, p->smem_bytes);
  if (p->occ_refill < 1) p->occ_refill = 1;
  if (p->occ_move < 1) p->occ_move = 1;
  if (p->occ_collide < 1) p->occ_collide = 1;
  p->pool_smem = pool_table_bytes(tl, p->use_smem) + pool_plane_bytes(geo->nx, geo->ny, geo->nz, M, G) + (size_t)POOL_WARPS * POOL_BYTES;
  bool attr_ok = p->use_smem != 0;      // the pool kernel keeps the cross-section tables in shared memory
  for (PoolFn f : POOL_VARIANTS)
    attr_ok = attr_ok && cudaFuncSetAttribute((const void *)f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->pool_smem) == cudaSuccess;
  if (!attr_ok) {
    cudaGetLastError(); p->pool_ok = 0;
  } else {
    p->occ_pool = 1 << 30;
    for (PoolFn f : POOL_VARIANTS) {
      int occ = 0;
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)f, POOL_THREADS, p->pool_smem);
      p->occ_pool = std::min(p->occ_pool, occ);
    }
    if (p->occ_pool < 1) p->pool_ok = 0;
  }
  p->pool = p->pool_ok;
  if (p->time_crossing && !p->pool_ok) {
    mcdc_problem_destroy(p);
    return fail(MCDC_EINVAL, "the time-crossing tally runs on the pool kernel, whose tables must fit in shared memory");
  }
  *out = p;
  return MCDC_OK;
}

extern "C" size_t mcdc_workspace_bytes(const mcdc_problem *p, const mcdc_run_params *rp)
{
  Layout L;
  if (!p || compute_layout(p, rp, &L) != MCDC_OK) return 0;
  return L.total;
}

extern "C" size_t mcdc_tally_size(const mcdc_problem *p) { return p ? p->n_tally : 0; }

extern "C" mcdc_status mcdc_run(mcdc_problem *p, const mcdc_run_params *rp, void *workspace_dev,
                                size_t workspace_bytes, void *cuda_stream)
{
  if (!p || !rp || !workspace_dev) return fail(MCDC_EINVAL, "null argument");
  Layout L;
  mcdc_status st = compute_layout(p, rp, &L);
  if (st != MCDC_OK) return st;
  if (workspace_bytes < L.total) return fail(MCDC_ENOMEM, "workspace too small: %zu < %zu", workspace_bytes, L.total);
  if (((uintptr_t)workspace_dev & 255) != 0) return fail(MCDC_EINVAL, "workspace must be 256-byte aligned");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  char *ws = (char *)workspace_dev;
  p->ran = false; p->ws = workspace_dev; p->lay = L; p->stream = s;
  p->n_batch = rp->n_batch; p->n_hist = rp->n_hist_per_batch;
  p->iterations = 0; p->launches = 0;
  if (const char *e = getenv("MCDC_MAX_FLIGHTS")) p->max_flights = atoi(e) > 0 ? atoi(e) : 1;
  if (const char *e = getenv("MCDC_TAIL")) p->tail_threshold = (uint64_t)atoll(e);
  if (const char *e = getenv("MCDC_FUSE_BULK")) p->fuse_bulk = atoi(e);
  if (const char *e = getenv("MCDC_REFILL")) p->refill = atoi(e);
  p->pool = p->pool_ok;
  if (const char *e = getenv("MCDC_POOL")) p->pool = (atoi(e) || p->time_crossing || p->eig_active > 0 || p->ic_on || p->dp.dn_J > 0 || p->dp.src_t1 > p->dp.src_t0) && p->pool_ok;
  const bool eig = p->eig_active > 0;
  if (eig && !p->pool) return fail(MCDC_EINVAL, "the eigenvalue mode runs on the pool kernel only");
  if (eig) p->k_cycle.assign((size_t)rp->n_batch * p->n_steps, 0.0);
  if (const char *e = getenv("MCDC_LONG_MFP")) p->long_mfp = atof(e);
  if (const char *e = getenv("MCDC_GROUP")) p->group = atoi(e) < 1 ? 1 : (atoi(e) > 4 ? 4 : atoi(e));
  p->prof_ms[0] = p->prof_ms[1] = 0.0; p->prof_launches[0] = p->prof_launches[1] = 0;

  struct PipeOut {
    uint64_t iterations = 0, launches = 0, prof_launches[2] = {0, 0};
    double prof_ms[2] = {0.0, 0.0};
    bool overflow = false;
    std::string err;
  } outs[4];
  std::atomic<uint32_t> next_batch{0u};
  std::mutex closeout_mu;
  const bool trace = p->profile && getenv("MCDC_TRACE") != nullptr;
  cudaStream_t s0 = s;
  {
    unsigned long long *d_cnt = (unsigned long long *)(ws + L.counters);
    double *sum1 = (double *)(ws + L.sum1), *sum2 = (double *)(ws + L.sum2);
    uint32_t *flag = (uint32_t *)(ws + L.flag);
    const uint32_t K = p->n_steps;
  CU(cudaMemsetAsync(d_cnt, 0, (size_t)rp->n_batch * K * N_CNT * 8, s0));
  CU(cudaMemsetAsync(sum1, 0, p->n_tally * 8, s0));
  CU(cudaMemsetAsync(sum2, 0, p->n_tally * 8, s0));
  CU(cudaMemsetAsync(flag, 0, 256, s0));

    CU(cudaStreamSynchronize(s0));
  }
  for (int i = 1; i < L.n_pipe; ++i)
    if (!p->aux_stream[i - 1]) CU(cudaStreamCreateWithFlags(&p->aux_stream[i - 1], cudaStreamNonBlocking));

  // One pipeline = one batch in flight: its own stream, control block, banks, queues and batch
  // tally.  Pipelines take batches from a shared counter; batch b always uses stream seed + b.
  auto pipe_main = [&](int pi) -> mcdc_status {
  PipeOut &po = outs[pi];
  cudaStream_t s = pi == 0 ? s0 : p->aux_stream[pi - 1];
  char *const pb = ws + L.pipe_base[pi];
  Ctl *ctl = (Ctl *)(pb + L.ctl);
  unsigned long long *d_cnt = (unsigned long long *)(ws + L.counters);
  double *tally = (double *)(pb + L.tally), *sum1 = (double *)(ws + L.sum1), *sum2 = (double *)(ws + L.sum2);
  const uint32_t cap = L.capacity;
  Bank bank[2] = { bank_at(pb, L.bankA, cap), bank_at(pb, L.bankB, cap) };
  Queues Q;
  Q.q[0] = (uint32_t *)(pb + L.q0); Q.q[1] = (uint32_t *)(pb + L.q1);
  Q.coll = (uint32_t *)(pb + L.qcoll); Q.census = (uint32_t *)(pb + L.qcensus);
  Q.capacity = cap;
  uint32_t *order = (uint32_t *)(pb + L.order), *bcount = (uint32_t *)(pb + L.bcount),
           *boffs = (uint32_t *)(pb + L.boffs), *bcursor = (uint32_t *)(pb + L.bcursor),
           *tiles = (uint32_t *)(pb + L.tiles), *flag = (uint32_t *)(ws + L.flag);
  uint32_t *const mirror_dev = p->host_mirror + 16 * pi;
  volatile uint32_t *mirror = mirror_dev;
  cudaEvent_t *const evp = p->ev + 12 * pi;
  DevProblem D = p->dp;
  D.tally = tally;
  const TableLayout tl = p->tl;
  const int use_smem = p->use_smem;
  const size_t smem = p->smem_bytes;
  const uint32_t K = p->n_steps;
  const uint64_t N = rp->n_hist_per_batch, M = comb_size(p, rp);
  const bool comb = M > 0 && K > 1;
  const bool wcomb = comb && p->ic_on;
  unsigned long long *wpre = (unsigned long long *)(pb + L.wpre), *wtiles = (unsigned long long *)(pb + L.wtiles);
  const uint32_t max_grid_move = (uint32_t)(p->sm_count * p->occ_move);
  uint32_t max_grid_refill = (uint32_t)(p->sm_count * p->occ_refill);
  if (L.n_pipe > 1) if (const char *e = getenv("MCDC_PIPE_DIV")) max_grid_refill = std::max(1u, max_grid_refill * 2u / (uint32_t)std::max(2, atoi(e)));
  // the persistent tail kernel keeps its blocks until its queue drains: with two pipelines each
  // takes half of the co-resident slots so that the other batch keeps running beside it
  const uint32_t max_grid_tail = std::max(1u, (uint32_t)(p->sm_count * p->occ_tail) / (uint32_t)L.n_pipe);
  const uint32_t max_grid_coll = (uint32_t)(p->sm_count * p->occ_collide);
  uint32_t max_grid_pool = (uint32_t)(p->sm_count * std::max(1, p->occ_pool));
  if (const char *e = getenv("MCDC_POOL_GRID")) max_grid_pool = std::max(1, atoi(e));
  const uint32_t max_grid = (uint32_t)p->sm_count * 8u;
  auto grid_for = [](uint64_t n, uint32_t mx) {
    uint64_t g = (n + BS - 1) / BS;
    return (uint32_t)(g < 1 ? 1 : (g > mx ? mx : g));
  };

  for (;;) {
    const uint32_t b = next_batch.fetch_add(1u);
    if (b >= rp->n_batch) break;
    const unsigned long long seedb = rp->seed + (unsigned long long)b;
    int cur = 0;                                     // bank holding the live particles
    CU(cudaMemsetAsync(tally, 0, p->n_tally * 8, s));
    k_begin_batch<<<1, 1, 0, s>>>(ctl, seedb, (uint32_t)N);
    k_source<<<grid_for(N, max_grid), BS, smem, s>>>(D, tl, use_smem, bank[cur], ctl, Q, (uint32_t)N);
    po.launches += 2;
    uint64_t n_active = N;
    double k_run = eig ? p->eig_k0 : 0.0;                // C.14: k the running generation is normalised with
    for (uint32_t k = 0; k < K; ++k) {
      if (eig && !(p->nu_max / k_run <= 7.0))
        return fail(MCDC_EINVAL, "cycle %u: fission yield nu/k = %g exceeds 7 children (k = %g)", k, p->nu_max / k_run, k_run);
      const double t_k = p->n_census > 0 ? p->t_census[k] : INFINITY;
      const bool last = (k == K - 1);
      k_begin_step<<<1, 1, 0, s>>>(ctl, t_k, last ? 1u : 0u, k + 1, d_cnt + ((size_t)b * K + k) * N_CNT,
                                   k == 0 ? (unsigned long long)N : 0ull, k_run,
                                   (!eig || (int)k >= p->eig_inactive) ? 1u : 0u);
      po.launches += 1;
      // event loop: one flight per active particle and iteration
      const uint32_t par0 = (uint32_t)(po.iterations & 1u);   // parity is 0 at the start of the step
      uint64_t tail_prev = (k == 0) ? (uint64_t)N : (uint64_t)mirror[3];
      if (p->pool) {
        // the whole census step in one persistent launch; relaunched only over fission children
        // that found the pools full (they sit behind the processed range of the active bank)
        k_pool_begin<<<1, 1, 0, s>>>(ctl, cap);
        po.launches += 1;
        while (n_active > 0) {
          const uint64_t want = (n_active + POOL_WARPS * 32 - 1) / (POOL_WARPS * 32);
          const uint32_t grid = (uint32_t)std::min<uint64_t>(max_grid_pool, std::max<uint64_t>(1, want));
          uint32_t chunk = n_active > (uint64_t)grid * POOL_WARPS * 512 ? 128u : 32u;
          if (const char *e = getenv("MCDC_POOL_CHUNK")) chunk = (uint32_t)std::max(32, atoi(e));
          if (p->profile) CU(cudaEventRecord(evp[0], s));
          pool_variant(p->time_crossing != 0, eig, p->ic_on != 0, p->dp.dn_J > 0 || p->dp.src_t1 > p->dp.src_t0)
              <<<grid, POOL_THREADS, p->pool_smem, s>>>(D, tl, use_smem, bank[cur], bank[cur ^ 1], ctl, Q, 0, chunk);
          if (p->profile) CU(cudaEventRecord(evp[1], s));
          k_pool_next<<<1, 1, 0, s>>>(ctl, mirror_dev, cap);
          po.launches += 2; po.iterations += 1;
          CU(cudaStreamSynchronize(s));
          if (p->profile) {
            float m0 = 0.f;
            CU(cudaEventElapsedTime(&m0, evp[0], evp[1])); po.prof_ms[0] += m0; po.prof_launches[0] += 1;
            if (trace)
              fprintf(stderr, "trace b%u k%u pool n_active=%llu grid=%u ms=%.4f -> spilled=%u n_census=%u flights=%llu\n",
                      b, k, (unsigned long long)n_active, grid, m0, mirror[0], mirror[1],
                      (unsigned long long)mirror[4] | ((unsigned long long)mirror[5] << 32));
          }
          n_active = mirror[0];
          if (mirror[2]) { po.overflow = true; n_active = 0; }
        }
        cur ^= 1;                                      // the census bank was written into the other bank
      }
      while (n_active > 0) {
        // long queues: event kernels (flights | collisions); short queues (the tail of a
        // census step): fused kernel that follows each particle to its end.  Very long
        // queues run a few iterations per host synchronisation (the kernels read the queue
        // lengths from the device control block; the host only needs them to pick the mode).
        const bool tail_mode = n_active <= p->tail_threshold;
        const bool fused = p->fuse_bulk || tail_mode;
        const int group = (!fused && p->refill && n_active > 8 * p->tail_threshold) ? p->group : 1;
        for (int gi = 0; gi < group; ++gi) {
          cudaEvent_t *ev = evp + 3 * gi;
          if (p->profile) CU(cudaEventRecord(ev[0], s));
          if (tail_mode) {
            // persistent tail: the next-queue buffer becomes the published part of the work queue
            const uint32_t par = (uint32_t)(po.iterations & 1u) ^ par0;
            CU(cudaMemsetAsync(Q.q[par ^ 1u], 0, (size_t)cap * 4, s));
            k_tail_begin<<<1, 1, 0, s>>>(ctl);
            k_flight<true, true><<<grid_for(2 * n_active, max_grid_tail), BS, smem, s>>>(D, tl, use_smem, bank[cur], ctl, Q, 1 << 30, 0u);
            po.launches += 1;
          } else if (fused)
            k_flight<true, false><<<grid_for(n_active, max_grid_move), BS, smem, s>>>(
                D, tl, use_smem, bank[cur], ctl, Q, p->max_flights, 0u);
          else if (p->refill)
            k_flight<false, false, true><<<std::min<uint32_t>(max_grid_refill, (uint32_t)((n_active + REFILL_THREADS - 1) / REFILL_THREADS)), REFILL_THREADS, smem, s>>>(
                D, tl, use_smem, bank[cur], ctl, Q, 1 << 30,
                n_active > (uint64_t)max_grid_refill * (REFILL_THREADS / 32) * 128 ? 128u : 32u);
          else
            k_flight<false, false><<<grid_for(n_active, max_grid_move), BS, smem, s>>>(
                D, tl, use_smem, bank[cur], ctl, Q, p->max_flights, 0u);
          if (p->profile) CU(cudaEventRecord(ev[1], s));
          if (!fused) {
            k_collide<<<grid_for(n_active, max_grid_coll), BS, smem, s>>>(D, tl, use_smem, bank[cur], ctl, Q);
            po.launches += 1;
          }
          if (p->profile) CU(cudaEventRecord(ev[2], s));
          k_flip<<<1, 1, 0, s>>>(ctl, mirror_dev);
          po.launches += 2; po.iterations += 1;
        }
        CU(cudaStreamSynchronize(s));
        if (p->profile) {
          for (int gi = 0; gi < group; ++gi) {
            cudaEvent_t *ev = evp + 3 * gi;
            float m0 = 0.f, m1 = 0.f;
            CU(cudaEventElapsedTime(&m0, ev[0], ev[1])); po.prof_ms[0] += m0; po.prof_launches[0] += 1;
            CU(cudaEventElapsedTime(&m1, ev[1], ev[2])); po.prof_ms[1] += m1; po.prof_launches[1] += 1;
            if (trace)
              fprintf(stderr, "trace b%u k%u it%llu n_active<=%llu fused=%d flight_ms=%.4f collide_ms=%.4f -> n_next=%u n_census=%u tail=%u flights=%llu\n",
                      b, k, (unsigned long long)po.iterations, (unsigned long long)n_active, (int)fused, m0, m1,
                      mirror[0], mirror[1], mirror[3], (unsigned long long)mirror[4] | ((unsigned long long)mirror[5] << 32));
          }
        }
        n_active = mirror[0];
        if (mirror[2]) { po.overflow = true; n_active = 0; }
        // fission chains: reclaim dead slots when the next iteration could exhaust the bank
        const uint64_t tail = mirror[3], live = n_active + mirror[1];
        const uint64_t growth = tail > tail_prev ? tail - tail_prev : 0;   // slots taken by the last iteration
        tail_prev = tail;
        if (n_active > 0 && tail + 4 * growth + n_active / 8 > cap && live < tail) {
          const uint32_t par = (uint32_t)(po.iterations & 1u) ^ par0;
          k_compact<<<grid_for(live, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], Q.q[par], Q.census, ctl);
          k_compact_done<<<1, 1, 0, s>>>(ctl, mirror_dev);
          po.launches += 2;
          cur ^= 1;
          tail_prev = live;
        }
      }
      if (po.overflow) break;                         // the census list is incomplete: no census close
      if (eig && !last) {
        // C.14: generation estimate of this cycle (children banked / generation size); it normalises
        // the next cycle.  (The last cycle's children are only counted: its estimate is filled in
        // from the census counter after the run.)
        const uint64_t n_f = mirror[1];
        k_run = k_run * (double)n_f / (double)N;
        p->k_cycle[(size_t)b * K + k] = k_run;
        if (n_f == 0) return fail(MCDC_ESTATE, "batch %u cycle %u: the fission source died out", b, k);
      }
      if (last) break;
      // census close: canonical order + comb, or hand the census list over
      if (comb) {
        BucketMap bm = L.bm;
        bm.base1 = (unsigned long long)k << 40;    // survivors alive in this step carry tag k
        CU(cudaMemsetAsync(bcount, 0, (size_t)bm.n_buckets * 4, s));
        const uint32_t gN = grid_for((uint64_t)cap, max_grid);
        k_bucket_hist<<<gN, BS, 0, s>>>(bm, bank[cur], Q.census, ctl, bcount, flag);
        k_scan_tiles<<<L.n_tiles, BS, 0, s>>>(bcount, bm.n_buckets, tiles);
        k_scan_sums<<<1, BS, 0, s>>>(tiles, L.n_tiles);
        k_scan_apply<<<L.n_tiles, BS, 0, s>>>(bcount, bm.n_buckets, tiles, boffs, bcursor);
        k_bucket_scatter<<<gN, BS, 0, s>>>(bm, bank[cur], Q.census, ctl, bcursor, order);
        k_bucket_sort<<<grid_for(bm.n_buckets, max_grid), BS, 0, s>>>(bank[cur], boffs, bcursor, bm.n_buckets, order);
        if (wcomb) {
          k_wq<<<gN, BS, 0, s>>>(bank[cur], order, ctl, wpre, flag);
          k_scan64_tiles<<<L.n_wtiles, BS, 0, s>>>(wpre, ctl, wtiles);
          k_scan64_sums<<<1, BS, 0, s>>>(wtiles, L.n_wtiles, ctl, wpre, flag);
          k_scan64_apply<<<L.n_wtiles, BS, 0, s>>>(wpre, ctl, wtiles);
          k_comb_weighted<<<grid_for(M, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], order, wpre, ctl, Q.q[0], M);
          po.launches += 4;
        } else {
        // groups with at least MCDC_LONG_MFP (64) mean free paths ahead of them in the next step go first
        const double dt_next = eig ? INFINITY : p->t_census[k + 1] - p->t_census[k];
        k_comb<<<grid_for(M, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], order, ctl, Q.q[0], M, p->vsig_dev,
                                                    p->long_mfp / dt_next, eig ? 1 : 0);
        }
        po.launches += 7;
        cur ^= 1;
      } else if (!p->pool) {                          // (the pool kernel writes the census bank densely itself)
        k_census_gather<<<grid_for((uint64_t)cap, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], Q.census, ctl, Q.q[0]);
        po.launches += 1;
        cur ^= 1;
      }
      k_end_step<<<1, 1, 0, s>>>(ctl, comb ? (unsigned long long)M : 0ull, mirror_dev, wcomb ? wpre : nullptr);
      po.launches += 1;
      CU(cudaStreamSynchronize(s));
      n_active = mirror[0];
      if (mirror[2]) po.overflow = true;
    }
    {                                               // one pipeline at a time folds into the shared sums
      std::lock_guard<std::mutex> lk(closeout_mu);
      k_closeout<<<grid_for(p->n_tally, max_grid), BS, 0, s>>>(tally, sum1, sum2, p->n_tally);
      po.launches += 1;
      if (b == rp->n_batch - 1)
        CU(cudaMemcpyAsync(ws + L.last, tally, p->n_tally * 8, cudaMemcpyDeviceToDevice, s));
      CU(cudaStreamSynchronize(s));
    }
  }
  uint32_t h_over = 0;
  CU(cudaMemcpy(&h_over, &ctl->overflow, 4, cudaMemcpyDeviceToHost));
  if (h_over) po.overflow = true;
  return MCDC_OK;
  };   // pipe_main
  // final state: overflow / uniform-weight flags, counters to the host
  int dev = 0;
  CU(cudaGetDevice(&dev));
  mcdc_status sts[4] = {MCDC_OK, MCDC_OK, MCDC_OK, MCDC_OK};
  std::vector<std::thread> ths;
  for (int i = 1; i < L.n_pipe; ++i)
    ths.emplace_back([&, i] { cudaSetDevice(dev); sts[i] = pipe_main(i); if (sts[i] != MCDC_OK) outs[i].err = g_err; });
  sts[0] = pipe_main(0);
  for (std::thread &t : ths) t.join();
  if (sts[0] != MCDC_OK) return sts[0];
  for (int i = 1; i < L.n_pipe; ++i) if (sts[i] != MCDC_OK) { g_err = outs[i].err; return sts[i]; }
  bool overflow = false;
  for (int i = 0; i < L.n_pipe; ++i) {
    p->iterations += outs[i].iterations; p->launches += outs[i].launches;
    for (int k2 = 0; k2 < 2; ++k2) { p->prof_ms[k2] += outs[i].prof_ms[k2]; p->prof_launches[k2] += outs[i].prof_launches[k2]; }
    overflow = overflow || outs[i].overflow;
  }
  const uint32_t K = p->n_steps;
  const uint32_t cap = L.capacity;
  uint32_t h_flag = 0, h_over = 0, h_flags[2] = {0, 0};
  CU(cudaMemcpyAsync(h_flags, ws + L.flag, 8, cudaMemcpyDeviceToHost, s));
  p->counters.assign((size_t)rp->n_batch * K * N_CNT, 0ull);
  CU(cudaMemcpyAsync(p->counters.data(), ws + L.counters, p->counters.size() * 8, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  CU(cudaGetLastError());
  p->ran = true;
  if (overflow || h_over) return fail(MCDC_EOVERFLOW, "particle bank capacity (%u slots) exceeded", cap);
  if (eig)
    for (uint32_t b = 0; b < rp->n_batch; ++b) {
      const double k_prev = K > 1 ? p->k_cycle[(size_t)b * K + K - 2] : p->eig_k0;
      const unsigned long long n_f = p->counters[((size_t)b * K + K - 1) * N_CNT + K_CENSUS];
      p->k_cycle[(size_t)b * K + K - 1] = k_prev * (double)n_f / (double)rp->n_hist_per_batch;
      if (n_f == 0) return fail(MCDC_ESTATE, "batch %u cycle %u: the fission source died out", b, K - 1);
    }
  h_flag = p->ic_on ? 0u : h_flags[0];
  if (h_flag) return fail(MCDC_EINVAL, "census bank weights are not uniform: the comb is defined for uniform weights");
  if (h_flags[1]) return fail(MCDC_EINVAL, "weighted comb: a weight outside [0, 2^19) or a total weight above 2^30");
  for (size_t r = 0; r < (size_t)rp->n_batch * K; ++r)
    if (p->counters[r * N_CNT + K_LOST]) return fail(MCDC_ELOST, "a particle left the tally mesh");
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_tally_read(const mcdc_problem *p, int which, double *out, size_t n, int out_is_device)
{
  if (!p || !out) return fail(MCDC_EINVAL, "null argument");
  if (!p->ran) return fail(MCDC_ESTATE, "mcdc_tally_read before mcdc_run");
  if (n != p->n_tally || which < 0 || which > 2) return fail(MCDC_EINVAL, "bad tally size or selector");
  char *ws = (char *)p->ws;
  cudaStream_t s = p->stream;
  const double *srcp;
  if (which == 2) srcp = (const double *)(ws + p->lay.last);
  else {
    double *dst = out_is_device ? out : (double *)(ws + p->lay.scratch);
    uint64_t g = (n + BS - 1) / BS; if (g > 148 * 8) g = 148 * 8; if (g < 1) g = 1;
    k_tally_stats<<<(uint32_t)g, BS, 0, s>>>((const double *)(ws + p->lay.sum1), (const double *)(ws + p->lay.sum2),
                                             dst, n, (double)p->n_batch,
                                             (double)p->n_hist * (p->eig_active > 0 ? (double)p->eig_active : 1.0), which);
    if (out_is_device) { CU(cudaStreamSynchronize(s)); return MCDC_OK; }
    srcp = dst;
  }
  CU(cudaMemcpyAsync(out, srcp, n * 8, out_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_counters_read(const mcdc_problem *p, uint32_t batch, int32_t step, mcdc_counters *out)
{
  if (!p || !out) return fail(MCDC_EINVAL, "null argument");
  if (!p->ran) return fail(MCDC_ESTATE, "mcdc_counters_read before mcdc_run");
  if (batch >= p->n_batch || step >= (int32_t)p->n_steps) return fail(MCDC_EINVAL, "batch or step out of range");
  unsigned long long acc[N_CNT] = {0};
  for (uint32_t k = 0; k < p->n_steps; ++k) {
    if (step >= 0 && (uint32_t)step != k) continue;
    const unsigned long long *c = &p->counters[((size_t)batch * p->n_steps + k) * N_CNT];
    for (int i = 0; i < N_CNT; ++i) acc[i] += c[i];
  }
  static_assert(sizeof(mcdc_counters) == N_CNT * 8, "counter layout");
  std::memcpy(out, acc, sizeof acc);
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_set_eigenvalue(mcdc_problem *p, int32_t n_inactive, int32_t n_active, double k0)
{
  if (!p) return fail(MCDC_EINVAL, "null argument");
  if (n_inactive < 0 || n_active < 1 || !(k0 > 0.0) || !std::isfinite(k0)) return fail(MCDC_EINVAL, "n_inactive >= 0, n_active >= 1, k0 > 0");
  if ((long long)n_inactive + n_active >= (1 << 22)) return fail(MCDC_EINVAL, "too many cycles");
  if (p->n_census != 0 || p->time_crossing) return fail(MCDC_EINVAL, "the eigenvalue mode is time-independent (n_census = 0, no time-crossing block)");
  if (p->ic_on) return fail(MCDC_EINVAL, "the eigenvalue mode is analog: not with implicit capture");
  if (p->dp.src_t1 > p->dp.src_t0) return fail(MCDC_EINVAL, "the eigenvalue mode is time-independent: not with a source window");
  if (!p->pool_ok) return fail(MCDC_EINVAL, "the eigenvalue mode runs on the pool kernel: the cross-section tables must fit in shared memory");
  p->eig_inactive = n_inactive; p->eig_active = n_active; p->eig_k0 = k0;
  p->n_steps = (uint32_t)(n_inactive + n_active);
  p->ran = false;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_set_implicit_capture(mcdc_problem *p, double w_roulette, double w_survive)
{
  if (!p) return fail(MCDC_EINVAL, "null argument");
  if (!(w_roulette >= 0.0) || (w_roulette > 0.0 && !(w_survive >= w_roulette)) || !(w_survive < 524288.0))
    return fail(MCDC_EINVAL, "0 <= w_roulette <= w_survive < 2^19 (w_roulette = 0: no roulette)");
  if (p->eig_active > 0) return fail(MCDC_EINVAL, "the eigenvalue mode is analog: not with implicit capture");
  if (!p->pool_ok) return fail(MCDC_EINVAL, "implicit capture runs on the pool kernel: the cross-section tables must fit in shared memory");
  p->ic_on = 1; p->dp.ic_w_roulette = w_roulette; p->dp.ic_w_survive = w_survive;
  p->ran = false;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_set_delayed(mcdc_problem *p, int32_t J, const double *nu_delayed, const double *decay,
                                        const double *chi_delayed)
{
  if (!p || !nu_delayed || !decay || !chi_delayed) return fail(MCDC_EINVAL, "null argument");
  if (J < 1 || J > 8) return fail(MCDC_EINVAL, "1 <= J <= 8 precursor groups");
  if (p->dp.dn_J > 0) return fail(MCDC_ESTATE, "delayed-neutron data already set");
  if (!p->pool_ok) return fail(MCDC_EINVAL, "delayed neutrons run on the pool kernel: the cross-section tables must fit in shared memory");
  const int M = p->dp.n_mat, G = p->dp.G;
  // the staged table block holds sigma_f and nu: read them back from the host copy
  const std::vector<double> &xs4 = p->host_xs4;
  std::vector<double> nup((size_t)M * G), cdf((size_t)M * J * G);
  for (int m = 0; m < M; ++m) {
    bool fissile = false;
    for (int g = 0; g < G; ++g) {
      double sd = 0.0;
      for (int j = 0; j < J; ++j) {
        const double x = nu_delayed[((size_t)m * G + g) * J + j];
        if (!(x >= 0.0)) return fail(MCDC_EINVAL, "negative delayed yield");
        sd = sd + x;
      }
      const double nu = xs4[(size_t)(m * G + g) * 4 + 3];
      if (sd > nu) return fail(MCDC_EINVAL, "delayed yields exceed nu (mat %d group %d)", m, g);
      nup[(size_t)m * G + g] = nu - sd;
      fissile = fissile || xs4[(size_t)(m * G + g) * 4 + 2] > 0.0;
    }
    for (int j = 0; j < J; ++j) {
      if (!(decay[m * J + j] > 0.0)) return fail(MCDC_EINVAL, "decay constants must be > 0");
      const double *row = chi_delayed + ((size_t)m * J + j) * G;
      double tot = 0.0;
      for (int g = 0; g < G; ++g) { if (!(row[g] >= 0.0)) return fail(MCDC_EINVAL, "negative delayed spectrum"); tot = tot + row[g]; }
      if (fissile && std::fabs(tot - 1.0) > 1e-12) return fail(MCDC_EINVAL, "delayed spectrum of material %d group %d does not sum to 1", m, j);
      build_cdf(row, G, tot, &cdf[((size_t)m * J + j) * G]);
    }
  }
  mcdc_status st = upload(p, nup.data(), nup.size(), &p->dp.dn_nup);
  if (st == MCDC_OK) st = upload(p, nu_delayed, (size_t)M * G * J, &p->dp.dn_nu);
  if (st == MCDC_OK) st = upload(p, decay, (size_t)M * J, &p->dp.dn_lambda);
  if (st == MCDC_OK) st = upload(p, cdf.data(), cdf.size(), &p->dp.dn_cdf);
  if (st != MCDC_OK) return st;
  p->dp.dn_J = J;
  p->ran = false;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_set_source_window(mcdc_problem *p, double t_end)
{
  if (!p) return fail(MCDC_EINVAL, "null argument");
  if (!(t_end > p->dp.src_t0) || !std::isfinite(t_end)) return fail(MCDC_EINVAL, "t_end must be finite and > t0");
  if (p->eig_active > 0) return fail(MCDC_EINVAL, "the eigenvalue mode is time-independent: not with a source window");
  if (!p->pool_ok) return fail(MCDC_EINVAL, "a source window runs on the pool kernel: the cross-section tables must fit in shared memory");
  p->dp.src_t1 = t_end;
  p->ran = false;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_keff_read(const mcdc_problem *p, uint32_t batch, double *k_cycle, size_t n)
{
  if (!p || !k_cycle) return fail(MCDC_EINVAL, "null argument");
  if (!p->ran) return fail(MCDC_ESTATE, "mcdc_keff_read before mcdc_run");
  if (p->eig_active < 1) return fail(MCDC_ESTATE, "not an eigenvalue run");
  if (batch >= p->n_batch || n != p->n_steps) return fail(MCDC_EINVAL, "batch out of range or n != n_inactive + n_active");
  std::memcpy(k_cycle, p->k_cycle.data() + (size_t)batch * p->n_steps, n * sizeof(double));
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_run_stats(const mcdc_problem *p, uint64_t *iterations, uint64_t *launches)
{
  if (!p) return fail(MCDC_EINVAL, "null argument");
  if (iterations) *iterations = p->iterations;
  if (launches) *launches = p->launches;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_kernel_path(const mcdc_problem *p, int *pool)
{
  if (!p || !pool) return fail(MCDC_EINVAL, "null argument");
  *pool = p->pool ? 1 : 0;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_profile(mcdc_problem *p, int enable)
{
  if (!p) return fail(MCDC_EINVAL, "null argument");
  if (enable) for (cudaEvent_t &e : p->ev) if (!e) CU(cudaEventCreate(&e));
  p->profile = enable ? 1 : 0;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_profile_read(const mcdc_problem *p, int kernel, double *ms, uint64_t *launches)
{
  if (!p || kernel < 0 || kernel > 1) return fail(MCDC_EINVAL, "kernel must be 0 (move) or 1 (collide)");
  if (ms) *ms = p->prof_ms[kernel];
  if (launches) *launches = p->prof_launches[kernel];
  return MCDC_OK;
}

// ---- measurement support: peak rate of no-return fp64 atomic adds (RED.ADD.F64) into an array of
// n_bins doubles at pseudo-random addresses (the denominator of the tally-atomic
// roofline is not published, so it is measured on the box).  arr_dev: device array of n_bins doubles.
namespace {
__global__ void __launch_bounds__(256) k_atomic_peak(double *arr, unsigned long long n_bins, unsigned long long n_ops)
{
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n_ops; i += stride) {
    unsigned long long h = i * 0x9E3779B97F4A7C15ull;      // Weyl/xorshift mix: spreads lanes over the array
    h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
    atomicAdd(arr + (h % n_bins), 1.0);
  }
}
}  // namespace

extern "C" mcdc_status mcdc_atomic_peak(void *arr_dev, uint64_t n_bins, uint64_t n_ops, void *cuda_stream, double *ms_out)
{
  if (!arr_dev || !n_bins || !n_ops || !ms_out) return fail(MCDC_EINVAL, "null argument");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  k_atomic_peak<<<148 * 8, 256, 0, s>>>((double *)arr_dev, n_bins, n_ops / 8);      // warm-up
  CU(cudaEventRecord(e0, s));
  k_atomic_peak<<<148 * 8, 256, 0, s>>>((double *)arr_dev, n_bins, n_ops);
  CU(cudaEventRecord(e1, s));
  CU(cudaEventSynchronize(e1));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *ms_out = ms;
  return MCDC_OK;
}
