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
#include <condition_variable>
#include <functional>
#include <mutex>
#include <thread>
#include <cstdlib>
#include <cstring>
#include <map>
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

constexpr int MAX_PIPE = 8;   // batches in flight at once, at most
struct Layout {          // byte offsets into the caller's workspace
  // shared by all pipelines (absolute offsets)
  size_t counters, last, sum1, sum2, scratch, flag, kcyc, total;
  // private to one pipeline (offsets relative to pipe_base[i])
  size_t ctl, tally, bankA, bankB, q0, q1, qcoll, qcensus, order, bcount, boffs, bcursor, tiles, wpre, wtiles, pipe_bytes;
  uint32_t n_wtiles;       // tiles of the 64-bit scan of the weighted comb
  size_t pipe_base[MAX_PIPE];
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
  std::vector<std::pair<void *, size_t>> dev_allocs;   // device blocks of the problem's tables (from / back to table_alloc)
  int n_census = 0;
  std::vector<double> t_census;
  uint64_t comb_target = 0;
  uint32_t n_steps = 1;
  size_t n_tally = 0;
  int sm_count = 0, occ_move = 2, occ_collide = 2, occ_tail = 1;
  uint32_t *host_mirror = nullptr;   // pinned, mapped: n_active, n_census, overflow, bank_tail (from a process-wide pool)
  // state of the last run
  bool ran = false;
  void *ws = nullptr;
  Layout lay{};
  cudaStream_t stream = nullptr;
  uint32_t n_batch = 0;
  uint32_t n_ranks = 1;              // replicas summed into the running sums (mcdc_replica_commit)
  uint64_t n_hist = 0;
  std::vector<unsigned long long> counters;  // [batch][step][16]
  uint64_t iterations = 0, launches = 0;
  // kernel-schedule switches of the parity tests, read ONCE from the environment at create (MCDC_POOL,
  // MCDC_PIPELINES, MCDC_POOL_GRID, MCDC_MARCH, MCDC_MAX_FLIGHTS, MCDC_TAIL, MCDC_FUSE_BULK, MCDC_REFILL); no result
  // depends on them
  int env_pool = -1;                 // -1: not set
  int env_pipelines = 0;             // 0: automatic
  int env_pool_grid = 0;             // 0: one block per co-resident slot
  int max_flights = 4;
  uint64_t tail_threshold = 0;       // set at create: 2 blocks of 256 lanes per SM
  int fuse_bulk = 0;
  int refill = 1;                    // persistent lanes refilled from the active queue (long queues)
  int occ_refill = 2;
  const double *vsig_dev = nullptr;  // [G] group speed x largest sigma_t of the group (comb: long histories first)
  int time_crossing = 0;             // the tally carries the time-crossing block (pool kernel only)
  int pool = 1;                      // one persistent pool launch per census step (mcdc_pool.cu)
  int pool_ok = 1;                   // the pool kernel can run this problem (tables fit in shared memory)
  // The variants that regroup tally marches (tally mesh finer than the lattice) pay off when a flight scores
  // several sub-segments: the choice follows the segments per flight the finished batches counted (results do
  // not depend on it; MCDC_MARCH = 0 | 1 fixes it for the parity tests).
  int march_ok = 0, march = 0, env_march = -1, occ_pool_march = 0;
  uint64_t table_hash = 0;           // key of g_march_learned
  int env_lean = 1;                  // MCDC_LEAN=0 (tests): the general kernel also where the lean variants apply
  int lean_ok = 0;                   // tally planes = lattice planes, no pins, tally time edges = census times (k_pool, POOL_LEAN)
  size_t pool_smem_march = 0;
  int occ_pool = 1;
  size_t pool_smem = 0;
  // k-eigenvalue mode (mcdc_set_eigenvalue; DESIGN.md §3 C.14): both 0 = fixed source
  int eig_inactive = 0, eig_active = 0;
  double eig_k0 = 1.0, nu_max = 0.0;
  std::vector<double> host_xs4;      // host copy of (sigma_t, sigma_s_row, sigma_f, nu) per (m, g)
  int ic_on = 0;                     // implicit capture + roulette + weighted comb (mcdc_set_implicit_capture; C.15)
  std::vector<double> k_cycle;       // [batch][cycle] generation estimate of k
  int profile = 0;
  cudaEvent_t ev[12 * 8] = {};         // per pipeline: 3 per iteration of a launch group
  double prof_ms[2] = {0.0, 0.0};        // k_move, k_collide
  uint64_t prof_launches[2] = {0, 0};
};

namespace {

// the instantiated variants of the pool kernel: <time-crossing, eigenvalue, implicit capture, delayed, march, csg>
using PoolFn = void (*)(DevProblem, TableLayout, int, Bank, Bank, Ctl *, Queues);
#define POOL_SET(MODE)                                                                                              \
    k_pool<false, false, false, false, MODE, false>, k_pool<true, false, false, false, MODE, false>, k_pool<false, true, false, false, MODE, false>, \
    k_pool<false, false, true, false, MODE, false>,  k_pool<true, false, true, false, MODE, false>,  k_pool<false, false, false, true, MODE, false>, \
    k_pool<true, false, false, true, MODE, false>,   k_pool<false, false, true, true, MODE, false>,  k_pool<true, false, true, true, MODE, false>,   \
    k_pool<false, true, false, true, MODE, false>
// quadric CSG (fixed-source modes, plain march): indexed by time-crossing | implicit capture << 1 | delayed << 2
#define POOL_CSG(TC, IC, DN) k_pool<TC, false, IC, DN, POOL_PLAIN, true>
const PoolFn POOL_VARIANTS[] = {POOL_SET(POOL_LEAN), POOL_SET(POOL_PLAIN), POOL_SET(POOL_MARCH),
                                POOL_CSG(false, false, false), POOL_CSG(true, false, false), POOL_CSG(false, true, false),
                                POOL_CSG(true, true, false),   POOL_CSG(false, false, true), POOL_CSG(true, false, true),
                                POOL_CSG(false, true, true),   POOL_CSG(true, true, true)};
#undef POOL_SET
#undef POOL_CSG
PoolFn pool_variant(bool tc, bool eig, bool ic, bool dn, int mode, bool csg)
{
  if (csg) return POOL_VARIANTS[30 + (tc ? 1 : 0) + (ic ? 2 : 0) + (dn ? 4 : 0)];
  const PoolFn *V = POOL_VARIANTS + 10 * mode;
  if (eig) return dn ? V[9] : V[2];
  if (dn && ic) return tc ? V[8] : V[7];
  if (dn) return tc ? V[6] : V[5];
  if (ic) return tc ? V[4] : V[3];
  return tc ? V[1] : V[0];
}

// ---- process-wide resources: what a problem needs from the CUDA runtime but need not own.  Creating
// them per problem (streams, a pinned mirror, function attributes, occupancy queries) cost more than
// the transfers of a create / run / read / destroy cycle.
std::mutex g_mu, g_run_mu;
size_t g_pool_smem_set = 0;                          // cudaFuncAttributeMaxDynamicSharedMemorySize of the pool variants
std::map<size_t, int> g_occ_pool;                    // dynamic shared memory -> blocks/SM (min over the variants)
struct EventOcc { int move, collide, tail, refill; };
std::map<size_t, EventOcc> g_occ_events;
cudaStream_t g_aux_stream[MAX_PIPE - 1] = {};          // streams of pipelines 1..7
cudaEvent_t g_ev_begin = nullptr, g_ev_done[MAX_PIPE - 1] = {};
std::vector<uint32_t *> g_mirror_free;               // 512-byte blocks of pinned mapped memory (16 words per pipeline)
// Host threads of pipelines 1..7: created once and kept (creating seven threads per mcdc_run cost 0.2 ms, a third of
// a step of config 1).  A worker sleeps on its condition variable between runs; the object is never destroyed (a
// thread blocked in a destroyed condition variable at exit would be undefined behaviour).
struct Worker {
  std::mutex m;
  std::condition_variable cv;
  std::function<void()> job;
  bool has_job = false, done = true, started = false;
};
Worker *g_workers = nullptr;          // [MAX_PIPE - 1], leaked on purpose; guarded by g_run_mu (one multi-pipeline run at a time)
void worker_main(Worker *w)
{
  for (;;) {
    std::function<void()> f;
    {
      std::unique_lock<std::mutex> lk(w->m);
      w->cv.wait(lk, [w] { return w->has_job; });
      f = std::move(w->job); w->has_job = false;
    }
    f();
    {
      std::lock_guard<std::mutex> lk(w->m);
      w->done = true;
    }
    w->cv.notify_all();
  }
}
void worker_start(int i, std::function<void()> f)
{
  if (!g_workers) g_workers = new Worker[MAX_PIPE - 1];
  Worker *w = g_workers + i;
  if (!w->started) { std::thread(worker_main, w).detach(); w->started = true; }
  {
    std::lock_guard<std::mutex> lk(w->m);
    w->job = std::move(f); w->has_job = true; w->done = false;
  }
  w->cv.notify_all();
}
void worker_wait(int i)
{
  Worker *w = g_workers + i;
  std::unique_lock<std::mutex> lk(w->m);
  w->cv.wait(lk, [w] { return w->done; });
}

// What a finished batch taught about a problem — whether its tally marches are long enough for the regrouped-march
// variants — is remembered under a hash of the problem's tables, so that the same problem created again (a caller
// that creates, runs and destroys per step: bench.py's e2e leg) starts with the variant it ended with.
std::map<uint64_t, int> g_march_learned;

// The attribute is per function and process-wide: it only ever grows, so that a problem created later
// with smaller tables cannot take the shared memory away from an earlier one.
bool pool_smem_ensure(size_t bytes)
{
  std::lock_guard<std::mutex> lk(g_mu);
  if (bytes <= g_pool_smem_set) return true;
  for (PoolFn f : POOL_VARIANTS)
    if (cudaFuncSetAttribute((const void *)f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) {
      cudaGetLastError();
      return false;
    }
  g_pool_smem_set = bytes;
  return true;
}
int pool_occupancy(size_t bytes)
{
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_occ_pool.find(bytes);
  if (it != g_occ_pool.end()) return it->second;
  int occ_min = 1 << 30;
  for (PoolFn f : POOL_VARIANTS) {
    int occ = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void *)f, POOL_THREADS, bytes);
    occ_min = std::min(occ_min, occ);
  }
  g_occ_pool[bytes] = occ_min;
  return occ_min;
}
EventOcc event_occupancy(size_t bytes)
{
  std::lock_guard<std::mutex> lk(g_mu);
  auto it = g_occ_events.find(bytes);
  if (it != g_occ_events.end()) return it->second;
  EventOcc o{1, 1, 1, 1};
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o.move, k_flight<false, false>, BS, bytes);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o.collide, k_collide, BS, bytes);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o.tail, k_flight<true, true>, BS, bytes);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o.refill, k_flight<false, false, true>, REFILL_THREADS, bytes);
  o.move = std::max(o.move, 1); o.collide = std::max(o.collide, 1); o.tail = std::max(o.tail, 1); o.refill = std::max(o.refill, 1);
  g_occ_events[bytes] = o;
  return o;
}
// Device blocks of problem tables are kept for the next problem instead of being freed (cudaFree synchronises the
// device; a create / destroy cycle per step is what the end-to-end measurement does): at most 8 blocks / 256 MB.
std::vector<std::pair<void *, size_t>> g_table_free;
size_t g_table_free_bytes = 0;
void *table_alloc(size_t bytes)
{
  {
    std::lock_guard<std::mutex> lk(g_mu);
    for (size_t i = 0; i < g_table_free.size(); ++i)
      if (g_table_free[i].second >= bytes && g_table_free[i].second <= 2 * bytes + 4096) {
        void *d = g_table_free[i].first;
        g_table_free_bytes -= g_table_free[i].second;
        g_table_free.erase(g_table_free.begin() + (long)i);
        return d;
      }
  }
  void *d = nullptr;
  if (cudaMalloc(&d, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return d;
}
void table_free(void *d, size_t bytes)
{
  {
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_table_free.size() < 8 && g_table_free_bytes + bytes <= ((size_t)256 << 20)) {
      g_table_free.emplace_back(d, bytes); g_table_free_bytes += bytes;
      return;
    }
  }
  cudaFree(d);
}
uint32_t *mirror_take()
{
  std::lock_guard<std::mutex> lk(g_mu);
  if (g_mirror_free.empty()) {
    uint32_t *blk = nullptr;
    if (cudaHostAlloc((void **)&blk, 4096, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    for (int i = 0; i < 8; ++i) g_mirror_free.push_back(blk + 128 * i);
  }
  uint32_t *m = g_mirror_free.back();
  g_mirror_free.pop_back();
  std::memset(m, 0, 256);
  return m;
}
void mirror_give(uint32_t *m)
{
  std::lock_guard<std::mutex> lk(g_mu);
  g_mirror_free.push_back(m);
}
mcdc_status aux_ensure(int n_pipe)
{
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_ev_begin) CU(cudaEventCreateWithFlags(&g_ev_begin, cudaEventDisableTiming));
  for (int i = 1; i < n_pipe; ++i) {
    if (!g_aux_stream[i - 1]) CU(cudaStreamCreateWithFlags(&g_aux_stream[i - 1], cudaStreamNonBlocking));
    if (!g_ev_done[i - 1]) CU(cudaEventCreateWithFlags(&g_ev_done[i - 1], cudaEventDisableTiming));
  }
  return MCDC_OK;
}

template <typename T>
mcdc_status upload(mcdc_problem *p, const T *host, size_t n, const T **dev)
{
  void *d = table_alloc((n ? n : 1) * sizeof(T));
  if (!d) return fail(MCDC_ECUDA, "cudaMalloc of %zu bytes failed", (n ? n : 1) * sizeof(T));
  p->dev_allocs.emplace_back(d, (n ? n : 1) * sizeof(T));
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
  L->kcyc = take((size_t)rp->n_batch * p->n_steps * 8);
  // batches in flight (MCDC_PIPELINES = 1..8): 2; 8 when a batch fills the pools only a few times (a launch
  // lasts as long as its longest history, so small batches leave most warps idle: measured on the
  // eigenvalue pin cell at 1e5 particles per cycle, 2.1e8 / 3.4e8 / 4.3e8 / 5.5e8 histories/s with 1 / 2 / 4 / 8, and at
  // 1e6 particles per batch +9 % (config 2), +9 % (config 3), +6 % (config 4) with 8 against 4)
  int np = nmax <= 2000000 ? MAX_PIPE : 2;
  if (p->env_pipelines) np = p->env_pipelines;
  np = (int)std::min<uint32_t>((uint32_t)np, rp->n_batch);
  L->n_pipe = np;
  for (int i = 0; i < MAX_PIPE; ++i) L->pipe_base[i] = off + (size_t)(i < np ? i : 0) * L->pipe_bytes;
  L->total = off + (size_t)np * L->pipe_bytes;
  return MCDC_OK;
}

Bank bank_at(char *base, size_t off, uint32_t cap)
{
  Bank B;
  char *p = base + off;
  B.xy.base = (double2 *)p; B.zt.base = B.xy.base + 1; B.uxy.base = B.xy.base + 2; B.uzw.base = B.xy.base + 3;
  p += (size_t)cap * 64;
  B.idp = (ulonglong2 *)p;
  return B;
}

__global__ void k_begin_batch(Ctl *ctl, unsigned long long seedb, uint32_t n_src, double eig_k0)
{
  ctl->n_active = n_src; ctl->n_next = 0; ctl->n_coll = 0; ctl->n_census = 0;
  ctl->bank_tail = n_src; ctl->parity = 0; ctl->overflow = 0; ctl->iter = 0;
  ctl->seedb = seedb;
  ctl->eig_k = eig_k0; ctl->spill_seen = 0; ctl->err_code = E_NONE; ctl->err_step = 0;
}

// eig_nu_max > 0: a generation of the eigenvalue mode (C.14); its yield nu / k must not exceed 7 children
__global__ void k_begin_step(Ctl *ctl, double t_k, uint32_t last, uint32_t k1, unsigned long long *cnt,
                             unsigned long long n_source, double eig_nu_max, uint32_t score)
{
  ctl->score = score;
  ctl->t_k = t_k; ctl->last_step = last; ctl->step_k1 = k1; ctl->cnt = cnt;
  ctl->n_census = 0; ctl->n_next = 0; ctl->n_coll = 0; ctl->parity = 0; ctl->fetch = 0;
  ctl->comb_front = 0; ctl->comb_back = 0;
  if (n_source) cnt[K_SOURCE] += n_source;
  if (eig_nu_max > 0.0 && !(eig_nu_max / ctl->eig_k <= 7.0)) {
    if (ctl->err_code == E_NONE) { ctl->err_code = E_EIG_YIELD; ctl->err_step = k1 - 1u; }
    ctl->n_active = 0u;                                  // nothing more is transported in this batch
  }
}

// after a census step: comb accounting (M > 0) or the census bank handed over as it is; in the eigenvalue
// mode (eig_N > 0) also the generation estimate k_c = k_{c-1} N_f / N (C.14), which normalises the next
// cycle.  N_f = children born in the cycle = its census counter (in the last cycle they are only counted).
__global__ void k_end_step(Ctl *ctl, unsigned long long M, uint32_t *mirror, const unsigned long long *w_pre,
                           unsigned long long eig_N, double *k_cycle, uint32_t last)
{
  const uint32_t n = ctl->n_census;
  if (eig_N && ctl->err_code == E_NONE && !ctl->overflow) {
    const unsigned long long n_f = ctl->cnt[K_CENSUS];
    const double k = ctl->eig_k * (double)n_f / (double)eig_N;
    ctl->eig_k = k; *k_cycle = k;
    if (n_f == 0ull) { ctl->err_code = E_EIG_DIED; ctl->err_step = ctl->step_k1 - 1u; }
  }
  if (!last) {
    if (ctl->overflow || ctl->err_code != E_NONE) { ctl->n_active = 0u; ctl->bank_tail = 0u; }
    else if (M) {
      ctl->cnt[K_COMB_IN] += n;
      // (weighted comb: a census bank of zero weights has no survivors)
      const bool out = n && !(w_pre && w_pre[n] == 0ull);
      if (out) ctl->cnt[K_COMB_OUT] += M;
      ctl->n_active = out ? (uint32_t)M : 0u;
      ctl->bank_tail = (uint32_t)M;
    } else { ctl->n_active = n; ctl->bank_tail = n; }
  }
  mirror[0] = ctl->n_active; mirror[1] = n; mirror[2] = ctl->overflow; mirror[3] = ctl->bank_tail;
  mirror[6] = ctl->spill_seen; mirror[7] = ctl->err_code; mirror[8] = ctl->err_step;
}

}  // namespace

extern "C" const char *mcdc_last_error(void) { return g_err.c_str(); }

extern "C" void mcdc_problem_destroy(mcdc_problem *p)
{
  if (!p) return;
  for (auto &d : p->dev_allocs) table_free(d.first, d.second);
  if (p->host_mirror) mirror_give(p->host_mirror);
  for (cudaEvent_t e : p->ev) if (e) cudaEventDestroy(e);
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
  if (src->kind < 0 || src->kind > 3) return fail(MCDC_EINVAL, "source kind");

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
  DevProblem &D = p->dp;
  D.n_mat = M; D.G = G;
  std::vector<double> vsig(G, 0.0);
  for (int g = 0; g < G; ++g) {
    double mx = 0.0;
    for (int m = 0; m < M; ++m) mx = std::max(mx, mat->sigma_t[m * G + g]);
    vsig[g] = mat->speed[g] * mx;
  }
  // every table goes into ONE device allocation, filled by one copy (a create / destroy pair costs one
  // cudaMalloc / cudaFree instead of fourteen)
  std::vector<unsigned char> pack;
  auto put = [&](const void *src, size_t bytes) {
    const size_t off = align256(pack.size());
    pack.resize(off + (bytes ? bytes : 1));
    if (bytes) std::memcpy(pack.data() + off, src, bytes);
    return off;
  };
  const size_t o_tab = put(tab.data(), tab.size() * 8);
  const size_t o_px = put(geo->xs, ((size_t)geo->nx + 1) * 8), o_py = put(geo->ys, ((size_t)geo->ny + 1) * 8),
               o_pz = put(geo->zs, ((size_t)geo->nz + 1) * 8);
  const size_t o_mo = put(mo.data(), nc), o_mi = put(mi.data(), nc), o_rad = put(geo->radius, nc * 8);
  const size_t o_vsig = put(vsig.data(), vsig.size() * 8), o_pins = put(pins.data(), pins.size() * sizeof(int));
  const size_t o_tx = put(tal->xs, ((size_t)tal->nx + 1) * 8), o_ty = put(tal->ys, ((size_t)tal->ny + 1) * 8),
               o_tz = put(tal->zs, ((size_t)tal->nz + 1) * 8), o_tt = put(tal->ts, ((size_t)tal->nt + 1) * 8);
  {
    uint64_t h = 1469598103934665603ull;               // FNV-1a over every table (cross sections, planes, maps, tally planes)
    for (unsigned char c : pack) { h ^= c; h *= 1099511628211ull; }
    p->table_hash = h;
  }
  char *dev = (char *)table_alloc(pack.size());
  if (!dev) { delete p; return fail(MCDC_ECUDA, "cudaMalloc of the problem tables (%zu bytes) failed", pack.size()); }
  p->dev_allocs.emplace_back(dev, pack.size());
  if (cudaMemcpy(dev, pack.data(), pack.size(), cudaMemcpyHostToDevice) != cudaSuccess) { mcdc_problem_destroy(p); cudaGetLastError(); return fail(MCDC_ECUDA, "copy of the problem tables failed"); }
  const double *dtab = (const double *)(dev + o_tab);
  D.xs4 = dtab + tl.xs4; D.cdf_s = dtab + tl.cdf_s; D.cdf_chi = dtab + tl.cdf_chi;
  D.cdf_src = dtab + tl.cdf_src; D.speed = dtab + tl.speed;
  D.nx = geo->nx; D.ny = geo->ny; D.nz = geo->nz;
  D.px = (const double *)(dev + o_px); D.py = (const double *)(dev + o_py); D.pz = (const double *)(dev + o_pz);
  D.mat_outer = (const int8_t *)(dev + o_mo); D.mat_inner = (const int8_t *)(dev + o_mi);
  D.radius = (const double *)(dev + o_rad);
  D.has_pins = pins.empty() ? 0 : 1;
  for (int i = 0; i < 6; ++i) D.bc[i] = geo->bc[i];
  D.src_kind = src->kind; D.src_isotropic = src->isotropic; D.src_t0 = src->t0; D.src_t1 = src->t0;
  for (int i = 0; i < 3; ++i) { D.src_lo[i] = src->lo[i]; D.src_hi[i] = src->hi[i]; D.src_dir[i] = src->dir[i]; }
  p->vsig_dev = (const double *)(dev + o_vsig);
  D.n_pins = (long long)pins.size();
  D.pin_cell = (const int *)(dev + o_pins);
  D.tnx = tal->nx; D.tny = tal->ny; D.tnz = tal->nz; D.tnt = tal->nt;
  D.tx = (const double *)(dev + o_tx); D.ty = (const double *)(dev + o_ty);
  D.tz = (const double *)(dev + o_tz); D.tt = (const double *)(dev + o_tt);
  D.tally = nullptr;
  auto hint = [](const double *t, int n) {
    AxisHint h{0.0, 0.0};
    if (std::isfinite(t[0]) && std::isfinite(t[n]) && t[n] > t[0]) { h.p0 = t[0]; h.inv_w = (double)n / (t[n] - t[0]); }
    return h;
  };
  auto same = [](const double *a, int na, const double *b, int nb) {
    return na == nb && std::memcmp(a, b, sizeof(double) * (size_t)(na + 1)) == 0;
  };
  D.planes_finite = std::isfinite(geo->xs[0]) && std::isfinite(geo->xs[geo->nx]) && std::isfinite(geo->ys[0]) &&
                    std::isfinite(geo->ys[geo->ny]) && std::isfinite(geo->zs[0]) && std::isfinite(geo->zs[geo->nz]);
  D.simple_tally = same(tal->xs, tal->nx, geo->xs, geo->nx) && same(tal->ys, tal->ny, geo->ys, geo->ny) &&
                   same(tal->zs, tal->nz, geo->zs, geo->nz);
  {
    // bins one census step / time bin keeps hot; with many more bins than lanes in flight two lanes of
    // a warp seldom meet in a bin (measured: DESIGN.md section 6)
    const size_t hot = (size_t)G * tal->nz * tal->ny * tal->nx;
    D.aggregate_tally = hot <= 4096 ? 1 : 0;
  }
  D.hx = hint(tal->xs, tal->nx); D.hy = hint(tal->ys, tal->ny);
  D.hz = hint(tal->zs, tal->nz); D.ht = hint(tal->ts, tal->nt);
  p->host_mirror = mirror_take();
  if (!p->host_mirror) { mcdc_problem_destroy(p); return fail(MCDC_ECUDA, "cudaHostAlloc failed"); }
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
  int devid = 0; cudaGetDevice(&devid);
  cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, devid);
  if (p->sm_count < 1) p->sm_count = 1;
  p->tail_threshold = (uint64_t)p->sm_count * 256 * 2;
  {
    const EventOcc o = event_occupancy(p->smem_bytes);
    p->occ_move = o.move; p->occ_collide = o.collide; p->occ_tail = o.tail; p->occ_refill = o.refill;
  }
  // a tally mesh finer than the lattice takes the kernel variants that can suspend and regroup tally marches
  D.march_min = MARCH_MIN; D.march_iter_min = MARCH_ITER_MIN; D.march_first = MARCH_FIRST;
  // (their tally plane tables are staged in shared memory: up to 16 KB of them)
  {
    // the lean kernel variants score one segment per flight in the time bin of the census step: every tally time
    // edge must be a census time (else flights that pass an edge inside a step would all take the slow march)
    bool t_same = tal->nt == std::max(cen->n_census, 1);
    for (int k = 0; t_same && k < tal->nt; ++k) {
      const double tk = cen->n_census > 0 ? cen->t_census[k] : INFINITY;
      t_same = std::memcmp(&tk, tal->ts + k + 1, sizeof(double)) == 0;
    }
    p->lean_ok = D.simple_tally && !D.has_pins && t_same;
  }
  p->march_ok = !D.simple_tally && tal->nx <= 65535 && tal->ny <= 65535 && tal->nz <= 65535 && tal->nt <= 65535 &&
             pool_tally_plane_bytes(tal->nx, tal->ny, tal->nz, tal->nt, true) <= 16 * 1024;
  p->pool_smem = pool_table_bytes(tl, p->use_smem) + pool_plane_bytes(geo->nx, geo->ny, geo->nz, M, G) +
                 (size_t)POOL_WARPS * pool_bytes(false);
  p->pool_smem_march = p->pool_smem + pool_tally_plane_bytes(tal->nx, tal->ny, tal->nz, tal->nt, true) + (size_t)POOL_WARPS * POOL_MARCH_BYTES;
  // the pool kernel keeps the cross-section tables in shared memory
  p->pool_ok = p->use_smem != 0 && pool_smem_ensure(p->pool_smem);
  if (p->pool_ok) {
    p->occ_pool = pool_occupancy(p->pool_smem);
    if (p->occ_pool < 1) p->pool_ok = 0;
  }
  if (p->pool_ok && p->march_ok) {
    p->occ_pool_march = pool_smem_ensure(p->pool_smem_march) ? pool_occupancy(p->pool_smem_march) : 0;
    if (p->occ_pool_march < 1) p->march_ok = 0;
  } else p->march_ok = 0;
  if (p->march_ok) {                                   // what an earlier problem with the same tables learned
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_march_learned.find(p->table_hash);
    if (it != g_march_learned.end()) p->march = it->second;
  }
  p->pool = p->pool_ok;
  // kernel-schedule switches of the parity tests (read once, here)
  if (const char *e = getenv("MCDC_POOL")) p->env_pool = atoi(e) ? 1 : 0;
  if (const char *e = getenv("MCDC_PIPELINES")) p->env_pipelines = std::min(MAX_PIPE, std::max(1, atoi(e)));
  if (const char *e = getenv("MCDC_POOL_GRID")) p->env_pool_grid = std::max(1, atoi(e));
  if (const char *e = getenv("MCDC_MARCH")) p->env_march = atoi(e) ? 1 : 0;
  if (const char *e = getenv("MCDC_LEAN")) p->env_lean = atoi(e);      // 0: general kernel; 2: lean kernel, every flight through its slow march
  if (const char *e = getenv("MCDC_MAX_FLIGHTS")) p->max_flights = atoi(e) > 0 ? atoi(e) : 1;
  if (const char *e = getenv("MCDC_TAIL")) p->tail_threshold = (uint64_t)atoll(e);
  if (const char *e = getenv("MCDC_FUSE_BULK")) p->fuse_bulk = atoi(e);
  if (const char *e = getenv("MCDC_REFILL")) p->refill = atoi(e);
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
  cudaStream_t s0 = (cudaStream_t)cuda_stream;
  char *ws = (char *)workspace_dev;
  p->ran = false; p->ws = workspace_dev; p->lay = L; p->stream = s0;
  p->n_batch = rp->n_batch; p->n_hist = rp->n_hist_per_batch; p->n_ranks = 1;
  p->iterations = 0; p->launches = 0;
  const bool eig = p->eig_active > 0;
  const bool needs_pool = p->time_crossing || eig || p->ic_on || p->dp.dn_J > 0 || p->dp.src_t1 > p->dp.src_t0 || p->dp.csg_n_region > 0;
  if (p->dp.src_kind == 3 && p->dp.csg_n_region == 0) return fail(MCDC_EINVAL, "the ball source (kind 3) belongs to the quadric CSG: call mcdc_set_csg");
  p->pool = p->pool_ok;
  if (p->env_pool >= 0) p->pool = (p->env_pool || needs_pool) && p->pool_ok;
  if (eig && !p->pool) return fail(MCDC_EINVAL, "the eigenvalue mode runs on the pool kernel only");
  if (p->pool && !pool_smem_ensure(std::max(p->pool_smem, p->march_ok ? p->pool_smem_march : 0) + pool_csg_bytes(p->dp.csg_n_surf)))
    return fail(MCDC_ECUDA, "cannot reserve %zu bytes of shared memory for the pool kernel", p->pool_smem);
  if (p->env_march >= 0) p->march = p->env_march && p->march_ok;
  const uint32_t K = p->n_steps;
  if (eig) p->k_cycle.assign((size_t)rp->n_batch * K, 0.0);
  p->prof_ms[0] = p->prof_ms[1] = 0.0; p->prof_launches[0] = p->prof_launches[1] = 0;

  struct PipeOut {
    uint64_t iterations = 0, launches = 0, prof_launches[2] = {0, 0};
    double prof_ms[2] = {0.0, 0.0};
    bool overflow = false;
    std::string err;
  } outs[MAX_PIPE];
  std::atomic<uint32_t> next_batch{0u};
  // (the other pipelines' streams and events are process-wide: runs that use them take turns)
  std::unique_lock<std::mutex> run_lk(g_run_mu, std::defer_lock);
  if (L.n_pipe > 1) run_lk.lock();
  std::mutex closeout_mu;
  uint32_t closeouts = 0;                              // (under closeout_mu) the first one writes the sums
  CU(cudaMemsetAsync(ws + L.counters, 0, (size_t)rp->n_batch * K * N_CNT * 8, s0));
  CU(cudaMemsetAsync(ws + L.flag, 0, 256, s0));
  if (eig) CU(cudaMemsetAsync(ws + L.kcyc, 0, (size_t)rp->n_batch * K * 8, s0));
  // the other pipelines' streams start after the caller's stream has reached this point
  st = aux_ensure(L.n_pipe);
  if (st != MCDC_OK) return st;
  if (L.n_pipe > 1) {
    CU(cudaEventRecord(g_ev_begin, s0));
    for (int i = 1; i < L.n_pipe; ++i) CU(cudaStreamWaitEvent(g_aux_stream[i - 1], g_ev_begin, 0));
  }

  // One pipeline = one batch in flight: its own stream, control block, banks, queues and batch
  // tally.  Pipelines take batches from a shared counter; batch b always uses stream seed + b.
  auto pipe_main = [&](int pi) -> mcdc_status {
  PipeOut &po = outs[pi];
  cudaStream_t s = pi == 0 ? s0 : g_aux_stream[pi - 1];
  char *const pb = ws + L.pipe_base[pi];
  Ctl *ctl = (Ctl *)(pb + L.ctl);
  unsigned long long *d_cnt = (unsigned long long *)(ws + L.counters);
  double *d_kcyc = (double *)(ws + L.kcyc);
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
  if (p->lean_ok && p->env_lean == 2) D.simple_tally = 2;
  const TableLayout tl = p->tl;
  const int use_smem = p->use_smem;
  const size_t smem = p->smem_bytes;
  const uint64_t N = rp->n_hist_per_batch, M = comb_size(p, rp);
  const bool comb = M > 0 && K > 1;
  const bool wcomb = comb && p->ic_on;
  unsigned long long *wpre = (unsigned long long *)(pb + L.wpre), *wtiles = (unsigned long long *)(pb + L.wtiles);
  const uint32_t max_grid_move = (uint32_t)(p->sm_count * p->occ_move);
  const uint32_t max_grid_refill = (uint32_t)(p->sm_count * p->occ_refill);
  // the persistent tail kernel keeps its blocks until its queue drains: with two pipelines each
  // takes half of the co-resident slots so that the other batch keeps running beside it
  const uint32_t max_grid_tail = std::max(1u, (uint32_t)(p->sm_count * p->occ_tail) / (uint32_t)L.n_pipe);
  const uint32_t max_grid_coll = (uint32_t)(p->sm_count * p->occ_collide);
  uint32_t grid_pool = 0;
  const uint32_t max_grid = (uint32_t)p->sm_count * 8u;
  auto grid_for = [](uint64_t n, uint32_t mx) {
    uint64_t g = (n + BS - 1) / BS;
    return (uint32_t)(g < 1 ? 1 : (g > mx ? mx : g));
  };
  PoolFn pool_fn = nullptr;
  size_t pool_smem = 0;
  // groups with at least 64 mean free paths ahead of them in the next census step are dealt in first
  constexpr double LONG_MFP = 64.0;

  // One batch.  waited = false (pool path only): every launch of the batch is queued without a host
  // round trip; kernels take the queue lengths from the device control block and launch shapes do not
  // depend on them.  The one thing the host would have to wait for — a relaunch of the pool kernel over
  // fission children that found the pools full — is rare (never in the five configs): the batch then
  // reports spill_seen and is run again with waited = true, which reproduces it exactly because every
  // draw is a function of (seed, id, flight counter).
  auto run_batch = [&](uint32_t b, bool waited, bool *again) -> mcdc_status {
    const unsigned long long seedb = rp->seed + (unsigned long long)b;
    int cur = 0;                                     // bank holding the live particles
    {
      const bool csg = p->dp.csg_n_region > 0;
      const bool march = p->march != 0 && !csg;      // (may change between batches: see below)
      // (the lean variants: tally planes = lattice planes and no pins, see k_pool)
      const int mode = march ? POOL_MARCH : (!csg && p->lean_ok && p->env_lean != 0) ? POOL_LEAN : POOL_PLAIN;
      pool_fn = pool_variant(p->time_crossing != 0, eig, p->ic_on != 0, p->dp.dn_J > 0 || p->dp.src_t1 > p->dp.src_t0, mode, csg);
      pool_smem = (march ? p->pool_smem_march : p->pool_smem) + (csg ? pool_csg_bytes(p->dp.csg_n_surf) : 0);
      // Blocks of the persistent launch.  One batch in flight: every co-resident slot.  Several: the launches of the
      // pipelines share the slots, so that one batch's tail (its last long histories) and its census close run beside
      // another batch's bulk instead of waiting for its blocks to retire: small batches (4 in flight) take 1 / n_pipe
      // of the slots each; two large batches take 7/8 each, which leaves room for the other's census-close kernels.
      // Measured: config 5 337 -> 327 ms per step; configs 1-4 +14 / +28 / +21 / +14 %.
      const uint32_t slots = (uint32_t)(p->sm_count * std::max(1, march ? p->occ_pool_march : p->occ_pool));
      const uint64_t nmax = std::max<uint64_t>(N, M);
      uint32_t share = slots;
      if (L.n_pipe >= 3 || (L.n_pipe == 2 && nmax <= 2000000)) share = slots / (uint32_t)L.n_pipe;
      else if (L.n_pipe == 2) share = slots - slots / 8u;
      grid_pool = p->env_pool_grid ? (uint32_t)p->env_pool_grid : std::max(1u, share);
    }
    CU(cudaMemsetAsync(tally, 0, p->n_tally * 8, s));
    k_begin_batch<<<1, 1, 0, s>>>(ctl, seedb, (uint32_t)N, eig ? p->eig_k0 : 0.0);
    k_source<<<grid_for(N, max_grid), BS, smem, s>>>(D, tl, use_smem, bank[cur], ctl, Q, (uint32_t)N);
    po.launches += 2;
    uint64_t n_active = N;
    for (uint32_t k = 0; k < K; ++k) {
      const double t_k = p->n_census > 0 ? p->t_census[k] : INFINITY;
      const bool last = (k == K - 1);
      k_begin_step<<<1, 1, 0, s>>>(ctl, t_k, last ? 1u : 0u, k + 1, d_cnt + ((size_t)b * K + k) * N_CNT,
                                   k == 0 ? (unsigned long long)N : 0ull, eig ? p->nu_max : 0.0,
                                   (!eig || (int)k >= p->eig_inactive) ? 1u : 0u);
      po.launches += 1;
      // event loop: one flight per active particle and iteration
      const uint32_t par0 = (uint32_t)(po.iterations & 1u);   // parity is 0 at the start of the step
      uint64_t tail_prev = (k == 0) ? (uint64_t)N : (uint64_t)mirror[3];
      if (p->pool) {
        // the whole census step in one persistent launch; relaunched only over fission children
        // that found the pools full (they sit behind the processed range of the active bank)
        k_pool_begin<<<1, 1, 0, s>>>(ctl, cap, grid_pool);
        po.launches += 1;
        do {
          if (p->profile) CU(cudaEventRecord(evp[0], s));
          pool_fn<<<grid_pool, POOL_THREADS, pool_smem, s>>>(D, tl, use_smem, bank[cur], bank[cur ^ 1], ctl, Q);
          if (cudaPeekAtLastError() != cudaSuccess)
            return fail(MCDC_ECUDA, "pool kernel launch failed: %s", cudaGetErrorString(cudaGetLastError()));
          if (p->profile) CU(cudaEventRecord(evp[1], s));
          k_pool_next<<<1, 1, 0, s>>>(ctl, mirror_dev, cap, grid_pool, waited ? 1u : 0u);
          po.launches += 2; po.iterations += 1;
          n_active = 0;
          if (waited || p->profile) {
            CU(cudaStreamSynchronize(s));
            if (p->profile) {
              float m0 = 0.f;
              CU(cudaEventElapsedTime(&m0, evp[0], evp[1])); po.prof_ms[0] += m0; po.prof_launches[0] += 1;
            }
            if (waited) {
              n_active = mirror[0];
              if (mirror[2]) { po.overflow = true; n_active = 0; }
            }
          }
        } while (n_active > 0);
        cur ^= 1;                                      // the census bank was written into the other bank
      }
      else while (n_active > 0) {
        // long queues: event kernels (flights | collisions); short queues (the tail of a
        // census step): fused kernel that follows each particle to its end.  Very long
        // queues run a few iterations per host synchronisation (the kernels read the queue
        // lengths from the device control block; the host only needs them to pick the mode).
        const bool tail_mode = n_active <= p->tail_threshold;
        const bool fused = p->fuse_bulk || tail_mode;
        const int group = (!fused && p->refill && n_active > 8 * p->tail_threshold) ? 4 : 1;
        for (int gi = 0; gi < group; ++gi) {
          cudaEvent_t *ev = evp + 3 * gi;
          if (p->profile) CU(cudaEventRecord(ev[0], s));
          if (tail_mode) {
            // persistent tail: the next-queue buffer becomes the published part of the work queue
            const uint32_t par = (uint32_t)(po.iterations & 1u) ^ par0;
            CU(cudaMemsetAsync(Q.q[par ^ 1u], 0, (size_t)cap * 4, s));
            k_tail_begin<<<1, 1, 0, s>>>(ctl);
            k_flight<true, true><<<grid_for(2 * n_active, max_grid_tail), BS, smem, s>>>(D, tl, use_smem, bank[cur], ctl, Q, 1 << 30, 0u);
            k_tail_spill<<<grid_for(n_active, max_grid), BS, 0, s>>>(ctl, Q);
            po.launches += 2;
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
      // census close: canonical order + comb, or hand the census list over
      if (!last && comb) {
        BucketMap bm = L.bm;
        bm.base1 = (unsigned long long)k << 40;    // survivors alive in this step carry tag k
        CU(cudaMemsetAsync(bcount, 0, (size_t)bm.n_buckets * 4, s));
        const uint32_t gN = grid_for((uint64_t)cap, max_grid);
        k_bucket_hist<<<gN, BS, 0, s>>>(bm, bank[cur], Q.census, ctl, bcount);
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
          const double dt_next = eig ? INFINITY : p->t_census[k + 1] - p->t_census[k];
          k_comb<<<grid_for(M, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], order, ctl, Q.q[0], M, p->vsig_dev,
                                                      LONG_MFP / dt_next, eig ? 1 : 0, flag);
        }
        po.launches += 7;
        cur ^= 1;
      } else if (!last && !p->pool) {                 // (the pool kernel writes the census bank densely itself)
        k_census_gather<<<grid_for((uint64_t)cap, max_grid), BS, 0, s>>>(bank[cur], bank[cur ^ 1], Q.census, ctl, Q.q[0]);
        po.launches += 1;
        cur ^= 1;
      }
      if (!last || eig) {
        k_end_step<<<1, 1, 0, s>>>(ctl, (comb && !last) ? (unsigned long long)M : 0ull, mirror_dev, wcomb ? wpre : nullptr,
                                   eig ? (unsigned long long)N : 0ull, d_kcyc + (size_t)b * K + k, last ? 1u : 0u);
        po.launches += 1;
      }
      if (last) break;
      if (waited || !p->pool) {
        CU(cudaStreamSynchronize(s));
        n_active = mirror[0];
        if (mirror[2]) po.overflow = true;
        if (mirror[7]) break;                          // (an error of the eigenvalue mode: reported below)
      } else n_active = 1;                             // (unknown to the host: the kernels read it from the control block)
    }
    {
      CU(cudaStreamSynchronize(s));                 // (the batch is complete: its flags decide whether it counts)
      uint32_t h[12] = {0};
      CU(cudaMemcpyAsync(h, &ctl->bank_tail, sizeof(uint32_t) * 3, cudaMemcpyDeviceToHost, s));   // bank_tail, parity, overflow
      uint32_t hs[3] = {0, 0, 0};
      CU(cudaMemcpyAsync(hs, &ctl->spill_seen, sizeof(uint32_t) * 3, cudaMemcpyDeviceToHost, s));  // spill_seen, err_code, err_step
      CU(cudaStreamSynchronize(s));
      if (h[2]) po.overflow = true;
      if (hs[0] && !waited && !po.overflow) { *again = true; return MCDC_OK; }
      if (po.overflow) return MCDC_OK;              // (reported for the whole run: MCDC_EOVERFLOW)
      if (p->pool && p->march_ok && p->env_march < 0 && p->dp.csg_n_region == 0) {
        // segments per flight of this batch decide which variant the following batches (and runs) take
        std::vector<unsigned long long> hc((size_t)K * N_CNT);
        CU(cudaMemcpy(hc.data(), d_cnt + (size_t)b * K * N_CNT, hc.size() * 8, cudaMemcpyDeviceToHost));
        unsigned long long fl = 0, sg = 0;
        for (uint32_t k2 = 0; k2 < K; ++k2) { fl += hc[(size_t)k2 * N_CNT + K_FLIGHTS]; sg += hc[(size_t)k2 * N_CNT + K_SEGMENTS]; }
        if (fl > 0) {
          p->march = (double)sg >= MARCH_SEGMENTS_PER_FLIGHT * (double)fl ? 1 : 0;
          std::lock_guard<std::mutex> lk(g_mu);
          g_march_learned[p->table_hash] = p->march;
        }
      }
      if (hs[1] == E_EIG_YIELD) {
        double kk = 0.0;
        if (hs[2] > 0) CU(cudaMemcpy(&kk, d_kcyc + (size_t)b * K + hs[2] - 1, 8, cudaMemcpyDeviceToHost)); else kk = p->eig_k0;
        return fail(MCDC_EINVAL, "cycle %u: fission yield nu/k = %g exceeds 7 children (k = %g)", hs[2], p->nu_max / kk, kk);
      }
      if (hs[1] == E_EIG_DIED) return fail(MCDC_ESTATE, "batch %u cycle %u: the fission source died out", b, hs[2]);
      std::lock_guard<std::mutex> lk(closeout_mu);  // one pipeline at a time folds into the shared sums
      k_closeout<<<grid_for(p->n_tally, max_grid), BS, 0, s>>>(tally, sum1, sum2, p->n_tally, closeouts == 0 ? 1 : 0);
      closeouts += 1;
      po.launches += 1;
      if (b == rp->n_batch - 1)
        CU(cudaMemcpyAsync(ws + L.last, tally, p->n_tally * 8, cudaMemcpyDeviceToDevice, s));
      CU(cudaStreamSynchronize(s));
    }
    return MCDC_OK;
  };   // run_batch

  for (;;) {
    const uint32_t b = next_batch.fetch_add(1u);
    if (b >= rp->n_batch) break;
    bool again = false;
    mcdc_status rs = run_batch(b, !p->pool, &again);
    if (rs == MCDC_OK && again) {
      // spilled children were left behind: the same batch once more, waiting for every pool launch
      CU(cudaMemsetAsync(d_cnt + (size_t)b * K * N_CNT, 0, (size_t)K * N_CNT * 8, s));
      rs = run_batch(b, true, &again);
    }
    if (rs != MCDC_OK) return rs;
    if (po.overflow) break;
  }
  return MCDC_OK;
  };   // pipe_main
  int dev = 0;
  CU(cudaGetDevice(&dev));
  mcdc_status sts[MAX_PIPE];
  for (mcdc_status &x : sts) x = MCDC_OK;
  for (int i = 1; i < L.n_pipe; ++i)
    worker_start(i - 1, [&, i] { cudaSetDevice(dev); sts[i] = pipe_main(i); if (sts[i] != MCDC_OK) outs[i].err = g_err; });
  sts[0] = pipe_main(0);
  for (int i = 1; i < L.n_pipe; ++i) worker_wait(i - 1);
  // the caller's stream continues after the other pipelines' streams
  for (int i = 1; i < L.n_pipe; ++i) {
    CU(cudaEventRecord(g_ev_done[i - 1], g_aux_stream[i - 1]));
    CU(cudaStreamWaitEvent(s0, g_ev_done[i - 1], 0));
  }
  if (sts[0] != MCDC_OK) return sts[0];
  for (int i = 1; i < L.n_pipe; ++i) if (sts[i] != MCDC_OK) { g_err = outs[i].err; return sts[i]; }
  bool overflow = false;
  for (int i = 0; i < L.n_pipe; ++i) {
    p->iterations += outs[i].iterations; p->launches += outs[i].launches;
    for (int k2 = 0; k2 < 2; ++k2) { p->prof_ms[k2] += outs[i].prof_ms[k2]; p->prof_launches[k2] += outs[i].prof_launches[k2]; }
    overflow = overflow || outs[i].overflow;
  }
  // final state: uniform-weight / fixed-point flags, counters (and the k of every cycle) to the host
  const uint32_t cap = L.capacity;
  uint32_t h_flags[2] = {0, 0};
  CU(cudaMemcpyAsync(h_flags, ws + L.flag, 8, cudaMemcpyDeviceToHost, s0));
  p->counters.assign((size_t)rp->n_batch * K * N_CNT, 0ull);
  CU(cudaMemcpyAsync(p->counters.data(), ws + L.counters, p->counters.size() * 8, cudaMemcpyDeviceToHost, s0));
  if (eig) CU(cudaMemcpyAsync(p->k_cycle.data(), ws + L.kcyc, p->k_cycle.size() * 8, cudaMemcpyDeviceToHost, s0));
  CU(cudaStreamSynchronize(s0));
  CU(cudaGetLastError());
  p->ran = true;
  if (overflow) return fail(MCDC_EOVERFLOW, "particle bank capacity (%u slots) exceeded", cap);
  if (!p->ic_on && h_flags[0]) return fail(MCDC_EINVAL, "census bank weights are not uniform: the comb is defined for uniform weights");
  if (h_flags[1]) return fail(MCDC_EINVAL, "weighted comb: a weight outside [0, 2^19) or a fixed-point total weight of 2^62 or more");
  for (size_t r = 0; r < (size_t)rp->n_batch * K; ++r)
    if (p->counters[r * N_CNT + K_LOST]) return fail(MCDC_ELOST, "a particle left the tally mesh or reached 2^24 - 1 flights");
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
    uint64_t g = (n + BS - 1) / BS; if (g > (uint64_t)p->sm_count * 8) g = (uint64_t)p->sm_count * 8; if (g < 1) g = 1;
    k_tally_stats<<<(uint32_t)g, BS, 0, s>>>((const double *)(ws + p->lay.sum1), (const double *)(ws + p->lay.sum2),
                                             dst, n, (double)p->n_batch * (double)p->n_ranks,
                                             (double)p->n_hist * (p->eig_active > 0 ? (double)p->eig_active : 1.0), which);
    if (out_is_device) { CU(cudaStreamSynchronize(s)); return MCDC_OK; }
    srcp = dst;
  }
  CU(cudaMemcpyAsync(out, srcp, n * 8, out_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_replica_layout(const mcdc_problem *p, size_t *sum1_offset, size_t *sum2_offset,
                                           size_t *counters_offset, size_t *counters_bytes)
{
  if (!p || !sum1_offset || !sum2_offset || !counters_offset || !counters_bytes) return fail(MCDC_EINVAL, "null argument");
  if (!p->ran) return fail(MCDC_ESTATE, "mcdc_replica_layout before mcdc_run");
  *sum1_offset = p->lay.sum1; *sum2_offset = p->lay.sum2; *counters_offset = p->lay.counters;
  *counters_bytes = (size_t)p->n_batch * p->n_steps * N_CNT * 8;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_replica_commit(mcdc_problem *p, uint32_t n_ranks)
{
  if (!p || n_ranks < 1) return fail(MCDC_EINVAL, "n_ranks >= 1");
  if (!p->ran) return fail(MCDC_ESTATE, "mcdc_replica_commit before mcdc_run");
  p->n_ranks = n_ranks;
  CU(cudaMemcpyAsync(p->counters.data(), (char *)p->ws + p->lay.counters, p->counters.size() * 8, cudaMemcpyDeviceToHost, p->stream));
  CU(cudaStreamSynchronize(p->stream));
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
  if (p->dp.csg_n_region > 0) return fail(MCDC_EINVAL, "the eigenvalue mode runs on the lattice geometry: not with mcdc_set_csg");
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

extern "C" mcdc_status mcdc_set_csg(mcdc_problem *p, int32_t n_surf, const double *coef, int32_t n_region,
                                    const int32_t *region_surf, const int32_t *region_mat)
{
  if (!p || !coef || !region_surf || !region_mat) return fail(MCDC_EINVAL, "null argument");
  if (p->dp.csg_n_region > 0) return fail(MCDC_ESTATE, "the quadric CSG is already set");
  if (n_surf < 1 || n_surf > 32 || n_region < 1 || n_region > 256) return fail(MCDC_EINVAL, "1 <= n_surf <= 32, 1 <= n_region <= 256");
  if (p->dp.nx != 1 || p->dp.ny != 1 || p->dp.nz != 1 || p->dp.has_pins)
    return fail(MCDC_EINVAL, "the quadric CSG divides ONE lattice cell without a pin (the cell's planes are the outer box)");
  if (p->eig_active > 0) return fail(MCDC_EINVAL, "the eigenvalue mode runs on the lattice geometry: not with mcdc_set_csg");
  if (!p->pool_ok) return fail(MCDC_EINVAL, "the quadric CSG runs on the pool kernel: the cross-section tables must fit in shared memory");
  std::vector<int8_t> rs((size_t)n_region * 8), rm(n_region);
  for (int q = 0; q < n_region; ++q) {
    if (region_mat[q] < 0 || region_mat[q] >= p->dp.n_mat) return fail(MCDC_EINVAL, "material of region %d out of range", q);
    rm[q] = (int8_t)region_mat[q];
    if (region_surf[q * 8] == 0) return fail(MCDC_EINVAL, "region %d has no surface", q);
    bool ended = false;
    for (int j = 0; j < 8; ++j) {
      const int e = region_surf[q * 8 + j];
      if (e == 0) ended = true;
      else if (ended) return fail(MCDC_EINVAL, "region %d: surface list with a gap", q);
      else if ((e > 0 ? e : -e) > n_surf) return fail(MCDC_EINVAL, "region %d: surface %d does not exist", q, e);
      rs[(size_t)q * 8 + j] = (int8_t)e;
    }
  }
  for (int i = 0; i < n_surf * 10; ++i) if (!std::isfinite(coef[i])) return fail(MCDC_EINVAL, "quadric coefficients must be finite");
  mcdc_status st = upload(p, coef, (size_t)n_surf * 10, &p->dp.csg_coef);
  if (st == MCDC_OK) st = upload(p, rs.data(), rs.size(), &p->dp.csg_rsurf);
  if (st == MCDC_OK) st = upload(p, rm.data(), rm.size(), &p->dp.csg_rmat);
  if (st != MCDC_OK) return st;
  if (!pool_smem_ensure(std::max(p->pool_smem, p->pool_smem_march) + pool_csg_bytes(n_surf)))
    return fail(MCDC_ECUDA, "cannot reserve the shared memory of the pool kernel with %d quadric surfaces", n_surf);
  p->dp.csg_n_surf = n_surf; p->dp.csg_n_region = n_region;
  p->ran = false;
  return MCDC_OK;
}

extern "C" mcdc_status mcdc_set_surface_motion(mcdc_problem *p, int32_t n_tau, const double *tau, const double *disp)
{
  if (!p || !tau || !disp) return fail(MCDC_EINVAL, "null argument");
  if (p->dp.csg_n_surf == 0) return fail(MCDC_ESTATE, "mcdc_set_surface_motion after mcdc_set_csg");
  if (p->dp.mv_n_tau > 0) return fail(MCDC_ESTATE, "the surface motion is already set");
  if (n_tau < 2 || n_tau > 32 || !ascending(tau, n_tau)) return fail(MCDC_EINVAL, "2 <= n_tau <= 32 strictly ascending break times");
  const int S = p->dp.csg_n_surf;
  for (int j = 0; j < n_tau; ++j) if (!std::isfinite(tau[j])) return fail(MCDC_EINVAL, "break times must be finite");
  for (int i = 0; i < S * n_tau * 3; ++i) if (!std::isfinite(disp[i])) return fail(MCDC_EINVAL, "displacements must be finite");
  // velocity of every interval: one divide per component (C.19); zero after the last break time
  std::vector<double> vel((size_t)S * n_tau * 3, 0.0);
  for (int s = 0; s < S; ++s)
    for (int k = 0; k + 1 < n_tau; ++k)
      for (int i = 0; i < 3; ++i)
        vel[((size_t)s * n_tau + k) * 3 + i] =
            (disp[((size_t)s * n_tau + k + 1) * 3 + i] - disp[((size_t)s * n_tau + k) * 3 + i]) / (tau[k + 1] - tau[k]);
  mcdc_status st = upload(p, tau, (size_t)n_tau, &p->dp.mv_tau);
  if (st == MCDC_OK) st = upload(p, disp, (size_t)S * n_tau * 3, &p->dp.mv_disp);
  if (st == MCDC_OK) st = upload(p, vel.data(), vel.size(), &p->dp.mv_vel);
  if (st != MCDC_OK) return st;
  p->dp.mv_n_tau = n_tau;
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

#include "mcdc_noalloc.cu"   // mcdc_batch_stats_noalloc: its own file-scope scratch array and entry point
