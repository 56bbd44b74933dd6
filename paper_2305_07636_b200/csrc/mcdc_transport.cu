// mcdc_transport.cu — event kernels of the history loop:
// table staging, source, move + track-length tally (+ surface and census dispatch),
// collision (capture / scatter / fission with secondary banking), queue compaction.
// Definitions: DESIGN.md §3.  sm_100a only; compiled with -fmad=false.
#include "mcdc_kernels.cuh"

namespace mcdc {

static __device__ __forceinline__ double d_inf() { return __longlong_as_double(0x7FF0000000000000ll); }

// ---- A0: stage the multigroup tables in shared memory ----------------------
struct Tables {
  const double *xs4, *cdf_s, *cdf_chi, *cdf_src, *speed;
};

static __device__ __forceinline__ Tables stage_tables(const DevProblem &P, const TableLayout &L,
                                                     double *smem, bool use_smem)
{
  Tables T;
  if (use_smem) {
    for (int i = threadIdx.x; i < L.total; i += blockDim.x) smem[i] = __ldg(P.xs4 + i);
    T.xs4 = smem + L.xs4; T.cdf_s = smem + L.cdf_s; T.cdf_chi = smem + L.cdf_chi;
    T.cdf_src = smem + L.cdf_src; T.speed = smem + L.speed;
  } else {
    T.xs4 = P.xs4; T.cdf_s = P.cdf_s; T.cdf_chi = P.cdf_chi; T.cdf_src = P.cdf_src; T.speed = P.speed;
  }
  return T;
}

// first j with xi < cdf[j] (the last entry is 1 > xi).  (Counting the entries <= xi without a
// data-dependent exit, looped or unrolled, was measured slower: most lanes stop at the first or
// second entry.)
static __device__ __forceinline__ int sample_cdf(const double *cdf, int n, double xi)
{
  int j = 0;
  while (j < n - 1 && !(xi < cdf[j])) ++j;
  return j;
}

// ---- counters: thread registers -> warp reduce -> shared -> one global atomic per block
static __device__ __forceinline__ void warp_count(unsigned long long *s_cnt, int slot, uint32_t v)
{
  const uint32_t tot = __reduce_add_sync(0xffffffffu, v);
  if ((threadIdx.x & 31) == 0 && tot) atomicAdd(&s_cnt[slot], (unsigned long long)tot);
}
static __device__ __forceinline__ void warp_count64(unsigned long long *s_cnt, int slot,
                                                    unsigned long long v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0 && v) atomicAdd(&s_cnt[slot], v);
}
static __device__ __forceinline__ void flush_counts(unsigned long long *s_cnt, unsigned long long *g_cnt)
{
  __syncthreads();
  if (threadIdx.x < N_CNT && s_cnt[threadIdx.x]) atomicAdd(&g_cnt[threadIdx.x], s_cnt[threadIdx.x]);
}

static __device__ __forceinline__ unsigned long long end_hash(uint64_t pid, uint32_t ectr, int ev)
{
  const U4 r = philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), ectr, BLK_FINGERPRINT + ev, 0u, 0u);
  return ((unsigned long long)r.x << 32) | (unsigned long long)r.y;
}

// ---- A13: block-level queue append: ballot/popc inside the warp, prefix over the
// warps in shared memory, ONE atomicAdd per block and queue.  cnt = entries this
// lane appends (0..3); returns the lane's first output position (valid if cnt>0).
static __device__ __forceinline__ uint32_t block_reserve(uint32_t cnt, uint32_t *counter,
                                                         uint32_t *s_w /*[NWARP+1]*/)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_w[wid] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < NWARP; ++w) { const uint32_t c = s_w[w]; s_w[w] = run; run += c; }
    s_w[NWARP] = run ? atomicAdd(counter, run) : 0u;
  }
  __syncthreads();
  const uint32_t pos = s_w[NWARP] + s_w[wid] + (incl - cnt);
  __syncthreads();
  return pos;
}

// exclusive prefix of cnt over the block and the block total (no atomic)
static __device__ __forceinline__ uint32_t block_scan_total(uint32_t cnt, uint32_t *s_w, uint32_t &total)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) s_w[wid] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < NWARP; ++w) { const uint32_t c = s_w[w]; s_w[w] = run; run += c; }
    s_w[NWARP] = run;
  }
  __syncthreads();
  const uint32_t pos = s_w[wid] + (incl - cnt);
  total = s_w[NWARP];
  __syncthreads();
  return pos;
}

// single-flag variant built on the warp ballot (the common case: 0/1 entries per lane)
static __device__ __forceinline__ uint32_t block_reserve1(bool flag, uint32_t *counter, uint32_t *s_w)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const uint32_t bal = __ballot_sync(0xffffffffu, flag);
  if (lane == 0) s_w[wid] = __popc(bal);
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < NWARP; ++w) { const uint32_t c = s_w[w]; s_w[w] = run; run += c; }
    s_w[NWARP] = run ? atomicAdd(counter, run) : 0u;
  }
  __syncthreads();
  const uint32_t pos = s_w[NWARP] + s_w[wid] + __popc(bal & ((1u << lane) - 1u));
  __syncthreads();
  return pos;
}

// ---- A6: warp-aggregated fp64 tally add (north_star item 6) ------------------
// All 32 lanes call it; bin < 0 = nothing to score.  Lanes hitting the same bin are
// found with __match_any_sync, summed with shuffles in ascending lane order, and the
// lowest lane issues one RED.ADD.F64.
static __device__ __forceinline__ double shfl_f64(double v, int src)
{
  int lo = __double2loint(v), hi = __double2hiint(v);
  lo = __shfl_sync(0xffffffffu, lo, src); hi = __shfl_sync(0xffffffffu, hi, src);
  return __hiloint2double(hi, lo);
}
static __device__ __forceinline__ void warp_tally_add(double *__restrict__ tally, long long bin, double val,
                                               bool aggregate = true)
{
  if (!aggregate) {                      // large tallies: same-bin lanes are rare, the match costs more than it saves
    if (bin >= 0) atomicAdd(tally + bin, val);
    return;
  }
  const int lane = threadIdx.x & 31;
  const unsigned peers = __match_any_sync(0xffffffffu, bin);
  if (__all_sync(0xffffffffu, peers == 0xffffffffu)) {       // one bin for the whole warp
    if (bin < 0) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) val += shfl_f64(val, lane ^ o);
    if (lane == 0) atomicAdd(tally + bin, val);
    return;
  }
  unsigned m = (bin >= 0) ? peers : 0u;
  const bool leader = m && (lane == __ffs(m) - 1);
  double acc = 0.0;
  while (__any_sync(0xffffffffu, m != 0u)) {
    const int src = m ? (__ffs(m) - 1) : lane;
    const double v = shfl_f64(val, src);
    if (m) { acc += v; m &= m - 1; }
  }
  if (leader) atomicAdd(tally + bin, acc);
}

// ---- A1: source sampling -----------------------------------------------------
__global__ void __launch_bounds__(BS) k_source(DevProblem P, TableLayout L, int use_smem, Bank B,
                                               Ctl *ctl, Queues Q, uint32_t n_src)
{
  extern __shared__ double smem[];
  const Tables T = stage_tables(P, L, smem, use_smem);
  __syncthreads();
  const unsigned long long seedb = ctl->seedb;
  for (uint32_t i = blockIdx.x * BS + threadIdx.x; i < n_src; i += gridDim.x * BS) {
    const uint64_t pid = i;
    const U4 rxy = draw_block(pid, 0, BLK_SRC_XY, seedb);
    const U4 rzg = draw_block(pid, 0, BLK_SRC_ZG, seedb);
    double ux, uy, uz;
    if (P.src_isotropic) {
      const U4 rd = draw_block(pid, 0, BLK_SRC_DIR, seedb);
      isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
    } else { ux = P.src_dir[0]; uy = P.src_dir[1]; uz = P.src_dir[2]; }
    double x, y, z;
    if (P.src_kind == 0) { x = P.src_lo[0]; y = P.src_lo[1]; z = P.src_lo[2]; }
    else if (P.src_kind == 1) {
      x = P.src_lo[0] + u52(rxy.x, rxy.y) * (P.src_hi[0] - P.src_lo[0]);
      y = P.src_lo[1] + u52(rxy.z, rxy.w) * (P.src_hi[1] - P.src_lo[1]);
      z = P.src_lo[2] + u52(rzg.x, rzg.y) * (P.src_hi[2] - P.src_lo[2]);
    } else if (P.src_kind == 3) {
      // C.18: uniform in the ball of centre src_lo and radius src_hi[0]: radius R max(xi1, xi2, xi3), isotropic
      // direction from the centre (the SRC_PIN block)
      const U4 rp = draw_block(pid, 0, BLK_SRC_PIN, seedb);
      double mx = u52(rxy.x, rxy.y);
      const double m2 = u52(rxy.z, rxy.w), m3 = u52(rzg.x, rzg.y);
      if (m2 > mx) mx = m2;
      if (m3 > mx) mx = m3;
      const double r = P.src_hi[0] * mx;
      double wx, wy, wz;
      isotropic_dir(u52(rp.x, rp.y), u52(rp.z, rp.w), wx, wy, wz);
      x = P.src_lo[0] + r * wx; y = P.src_lo[1] + r * wy; z = P.src_lo[2] + r * wz;
    } else {
      const U4 rp = draw_block(pid, 0, BLK_SRC_PIN, seedb);
      long long pin = (long long)(u52(rp.x, rp.y) * (double)P.n_pins);
      if (pin > P.n_pins - 1) pin = P.n_pins - 1;
      const int c = P.pin_cell[pin];
      const int cix = c % P.nx, ciy = (c / P.nx) % P.ny;
      const double cx = 0.5 * (P.px[cix] + P.px[cix + 1]), cy = 0.5 * (P.py[ciy] + P.py[ciy + 1]);
      const double rho = P.radius[c] * sqrt(u52(rp.z, rp.w));
      double cs, sn;
      mc_sincos2pi(u52(rxy.x, rxy.y), cs, sn);
      x = cx + rho * cs; y = cy + rho * sn;
      z = P.src_lo[2] + u52(rzg.x, rzg.y) * (P.src_hi[2] - P.src_lo[2]);
    }
    const int g = sample_cdf(T.cdf_src, P.G, u52(rzg.z, rzg.w));
    const int ix = find_interval(P.px, P.nx, x, ux);
    const int iy = find_interval(P.py, P.ny, y, uy);
    const int iz = find_interval(P.pz, P.nz, z, uz);
    int inside = 0;
    const int c = (iz * P.ny + iy) * P.nx + ix;
    if (P.has_pins && P.mat_inner[c] >= 0) {
      const double cx = 0.5 * (P.px[ix] + P.px[ix + 1]), cy = 0.5 * (P.py[iy] + P.py[iy + 1]);
      const double dx = x - cx, dy = y - cy, R = P.radius[c];
      inside = fma(dx, dx, dy * dy) < R * R;
    }
    B.xy[i] = make_double2(x, y);
    double t_birth = P.src_t0;
    if (P.src_t1 > P.src_t0) {                     // C.17
      const U4 rt = draw_block(pid, 0, BLK_SRC_TIME, seedb);
      t_birth = P.src_t0 + u52(rt.x, rt.y) * (P.src_t1 - P.src_t0);
    }
    B.zt[i] = make_double2(z, t_birth);
    B.uxy[i] = make_double2(ux, uy);
    B.uzw[i] = make_double2(uz, 1.0);
    int ixr = ix;
    if (P.csg_n_region > 0) {                       // C.18: the region travels in the ix field (the box is cell 0)
      const int r = find_region(P, P.csg_coef, -1, -1, x, y, z, t_birth);
      ixr = r < 0 ? CSG_NO_REGION : r;
    }
    B.idp[i] = make_ulonglong2(pid, pack_state(0, g, ixr, iy, iz, inside));
    Q.q[0][i] = i;
  }
}

// ---- A3-A7, A11 (+ A8-A10 when FUSE): flights of the active particles --------------
// Each lane carries one particle through up to max_flights consecutive flights:
// distances, event select, warp-synchronous tally march, move/snap, surface and census
// dispatch in registers.  Without FUSE a collision ends the lane's work (the particle
// is queued for k_collide); with FUSE the collision is resolved in place (the lane
// adopts the first fission child, further children are banked with atomic appends),
// which is how the short-queue tail of a census step is drained in few launches.
struct Lane {
  double x, y, z, t, ux, uy, uz, w;
  uint64_t pid;
  uint32_t ectr;
  int g, ix, iy, iz, inside;
  int m, pin;            // material of the current region; pin material of the cell (-1: none)
};

// material lookup when the particle enters a cell / region: issued at the END of a flight so
// that the dependent load overlaps the bookkeeping and the random draw of the next one
static __device__ __forceinline__ void lane_material(const DevProblem &P, Lane &p)
{
  const int cell = (p.iz * P.ny + p.iy) * P.nx + p.ix;
  p.pin = P.has_pins ? (int)__ldg(P.mat_inner + cell) : -1;
  p.m = p.inside ? p.pin : (int)__ldg(P.mat_outer + cell);
}

// WQ (with FUSE): the tail of a census step as ONE persistent launch over a device-side
// work queue.  Idle lanes take tickets (atomic head); tickets below n address the active
// queue, later tickets address entries that running lanes publish (slot + 1, written
// after a __threadfence) when a fission banks further children, so a family spreads over
// the idle lanes instead of serialising on one.  wq_pending counts unfinished particles;
// a lane leaves when it holds an unfilled ticket and wq_pending is 0.
static __device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t *p)
{
  return *(const volatile uint32_t *)p;
}

// Bank slots of particles that end inside the tail kernel are recycled by the lane that
// saw them end: a few spare slots per lane serve its next fission children / census
// copies before the bank tail is bumped (no cross-lane free list: no extra atomics).
constexpr int N_SPARE = 4;
// blocks per SM the register allocation aims at (measured: the refill kernel is faster without
// spills at 2 blocks/SM than with them at 3)
#ifndef MB_REFILL
#define MB_REFILL 2
#endif
#ifndef REFILL_THREADS
#define REFILL_THREADS 256      // the refill kernel has no block-wide step: its block size is free
#endif
#ifndef MB_WQ
#define MB_WQ 2
#endif
#ifndef MB_COLLIDE
#define MB_COLLIDE 3
#endif
#ifndef MB_PLAIN
#define MB_PLAIN 3
#endif

// REFILL (long queues): persistent warps keep every lane busy.  A lane whose particle
// leaves the flight loop (collision, census, end) hands it in and takes the next entry of
// the active queue in the same round: warps reserve chunks of the queue with one atomic
// (Ctl::fetch) and deal them to their idle lanes by ballot; finished particles are staged
// per warp in shared memory and appended to the collision / census lists in bursts (one
// atomic per burst).  No block-wide barrier inside the loop.
static __device__ __forceinline__ void stage_flush(const uint32_t *buf, uint32_t cnt, uint32_t *counter,
                                                   uint32_t *__restrict__ list)
{
  if (cnt == 0u) return;                       // cnt is warp-uniform
  const int lane = threadIdx.x & 31;
  uint32_t b = 0;
  if (lane == 0) b = atomicAdd(counter, cnt);
  b = __shfl_sync(0xffffffffu, b, 0);
  for (uint32_t k = lane; k < cnt; k += 32) list[b + k] = buf[k];
  __syncwarp();
}
constexpr int STAGE_CAP = 96, STAGE_FLUSH = 64;

template <bool FUSE, bool WQ, bool REFILL = false>
__global__ void __launch_bounds__(REFILL ? REFILL_THREADS : BS, REFILL ? MB_REFILL : (WQ ? MB_WQ : MB_PLAIN)) k_flight(DevProblem P, TableLayout L, int use_smem, Bank B,
                                               Ctl *ctl, Queues Q, int max_flights, uint32_t fetch_chunk)
{
  extern __shared__ double smem[];
  __shared__ uint32_t s_w[NWARP + 1];
  __shared__ unsigned long long s_cnt[N_CNT];
  __shared__ uint32_t s_stage[REFILL ? NWARP : 1][2][REFILL ? STAGE_CAP : 1];
  const Tables T = stage_tables(P, L, smem, use_smem);
  if (threadIdx.x < N_CNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const uint32_t n = ctl->n_active;
  const uint32_t par = ctl->parity;
  const uint32_t *__restrict__ q_in = Q.q[par];
  uint32_t *__restrict__ q_out = Q.q[par ^ 1u];
  const double t_k = ctl->t_k;
  const unsigned long long seedb = ctl->seedb;
  const bool last_step = ctl->last_step != 0u;
  const double INF = d_inf();
  const int G = P.G;
  // simple-tally path: time bin of this census step and the 32-bit strides of the bin index
  int jt_step = -1;
  if (P.simple_tally) {
    int lo = 0, hi = P.tnt;                        // first edge index j+1 with tt[j+1] >= t_k
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(P.tt + mid) < t_k) lo = mid; else hi = mid; }
    if (__ldg(P.tt + lo + 1) == t_k) jt_step = lo;
    else if (__ldg(P.tt + 1) == t_k) jt_step = 0;
  }
  const double t_lo_step = jt_step >= 0 ? __ldg(P.tt + jt_step) : 0.0;
  const int g_stride = P.tnz * P.tny * P.tnx;
  const bool small_tally = (long long)g_stride * G < (1ll << 30);
  if (!small_tally) jt_step = -1;                  // (keeps the in-bin arithmetic in 32 bits)
  const long long bin_t0 = (long long)(jt_step >= 0 ? jt_step : 0) * G * g_stride;

  uint32_t c_flights = 0, c_segments = 0, c_cross = 0, c_refl = 0, c_leak = 0, c_census = 0, c_lost = 0;
  uint32_t c_coll = 0, c_scat = 0, c_capt = 0, c_fis = 0, c_sec = 0;
  unsigned long long fp = 0ull;

  for (uint32_t base = blockIdx.x * BS; (WQ || REFILL) ? base == blockIdx.x * BS : base < n; base += gridDim.x * BS) {
    const uint32_t i = base + threadIdx.x;
    const bool valid = !WQ && !REFILL && i < n;
    uint32_t slot = 0;
    Lane p;
    p.x = p.y = p.z = p.t = 0.0; p.ux = 1.0; p.uy = p.uz = 0.0; p.w = 0.0;
    p.pid = 0; p.ectr = 0; p.g = 0; p.ix = p.iy = p.iz = 0; p.inside = 0; p.m = 0; p.pin = -1;
    if (valid) {
      slot = q_in[i];
      const double2 a = B.xy[slot], b = B.zt[slot], c2 = B.uxy[slot], e2 = B.uzw[slot];
      const ulonglong2 id = B.idp[slot];
      p.x = a.x; p.y = a.y; p.z = b.x; p.t = b.y; p.ux = c2.x; p.uy = c2.y; p.uz = e2.x; p.w = e2.y;
      p.pid = id.x;
      p.ectr = pk_ectr(id.y); p.g = pk_g(id.y); p.ix = pk_ix(id.y); p.iy = pk_iy(id.y);
      p.iz = pk_iz(id.y); p.inside = pk_inside(id.y);
      lane_material(P, p);
    }
    bool live = valid, dir_dirty = false;
    int outcome = 0;                  // 0 dead, 1 next flight, 2 collision queue, 3 census bank
    int nfl = 0;
    bool slot_free = true;            // WQ: the particle's own bank slot can take its census copy
    bool done = !(WQ || REFILL), has_ticket = false;
    // REFILL: the warp's reserved range of the active queue and its staged output lists
    uint32_t rng_next = 0, rng_end = 0, n_st_coll = 0, n_st_cens = 0;
    bool exhausted = false;
    const int lane_id = threadIdx.x & 31, warp_id = threadIdx.x >> 5;
    const unsigned lt_mask = (1u << lane_id) - 1u;
    uint32_t ticket = 0, idle_polls = 0, wq_round = 0;
    uint32_t spare[N_SPARE]; int nsp = 0;

    while (__any_sync(0xffffffffu, live || !done)) {
      double d = 0.0, v = 1.0, sig_t = 1.0;
      int ev = 0, surf = 0, m = 0;
      if (REFILL) {
        const unsigned need = __ballot_sync(0xffffffffu, !live);
        if (need && !exhausted) {
          if (rng_next == rng_end) {                      // reserve the next chunk of the active queue
            uint32_t b = 0;
            if (lane_id == 0) b = atomicAdd(&ctl->fetch, fetch_chunk);
            b = __shfl_sync(0xffffffffu, b, 0);
            rng_next = min(b, n); rng_end = min(b + fetch_chunk, n);
            if (rng_next == rng_end) exhausted = true;
          }
          if (!exhausted) {
            const uint32_t my = rng_next + __popc(need & lt_mask);
            if (!live && my < rng_end) {
              slot = q_in[my];
              const double2 a = B.xy[slot], b = B.zt[slot], c2 = B.uxy[slot], e2 = B.uzw[slot];
              const ulonglong2 id = B.idp[slot];
              p.x = a.x; p.y = a.y; p.z = b.x; p.t = b.y; p.ux = c2.x; p.uy = c2.y; p.uz = e2.x; p.w = e2.y;
              p.pid = id.x;
              p.ectr = pk_ectr(id.y); p.g = pk_g(id.y); p.ix = pk_ix(id.y); p.iy = pk_iy(id.y);
              p.iz = pk_iz(id.y); p.inside = pk_inside(id.y);
              lane_material(P, p);
              live = true; dir_dirty = false; outcome = 0; nfl = 0;
            }
            rng_next = min(rng_end, rng_next + (uint32_t)__popc(need));
          }
        }
        done = exhausted;
        if (!__any_sync(0xffffffffu, live)) { if (exhausted) break; continue; }
      }
      // (the overflow flag and the tickets are polled every 4th round only: their L2 round trip
      // would otherwise sit on the critical path of the lanes that are flying)
      if (WQ && (wq_round++ & 3u) == 0u) {
      if (ld_volatile_u32(&ctl->overflow) != 0u) { live = false; done = true; }   // run is invalid: stop
      if (!live && !done) {       // idle lane: take / poll a ticket of the work queue
        if (!has_ticket) { ticket = atomicAdd(&ctl->wq_head, 1u); has_ticket = true; }
        bool got = false;
        if (ticket < n) { slot = q_in[ticket]; got = true; }
        else if (ticket - n < Q.capacity) {
          const uint32_t e = ld_volatile_u32(q_out + (ticket - n));
          if (e) { slot = e - 1u; got = true; }
        }
        if (got) {
          __threadfence();
          const double2 a = __ldcg(B.xy + slot), b = __ldcg(B.zt + slot), c2 = __ldcg(B.uxy + slot),
                        e2 = __ldcg(B.uzw + slot);
          const ulonglong2 id = __ldcg(B.idp + slot);
          p.x = a.x; p.y = a.y; p.z = b.x; p.t = b.y; p.ux = c2.x; p.uy = c2.y; p.uz = e2.x; p.w = e2.y;
          p.pid = id.x;
          p.ectr = pk_ectr(id.y); p.g = pk_g(id.y); p.ix = pk_ix(id.y); p.iy = pk_iy(id.y);
          p.iz = pk_iz(id.y); p.inside = pk_inside(id.y);
          lane_material(P, p);
          live = true; has_ticket = false; slot_free = true; idle_polls = 0;
        } else if (ld_volatile_u32(&ctl->wq_pending) == 0u) done = true;
        else if (++idle_polls > (1u << 25)) { atomicExch(&ctl->overflow, 2u); done = true; }   // safety valve
      }
      }
      if (WQ && !__any_sync(0xffffffffu, live)) { __nanosleep(200); continue; }
      const bool was_live = live;
      int end_ev = -1; uint64_t end_pid = 0; uint32_t end_ectr = 0;   // terminal event of this flight, hashed below
      if (live) {
        const int pin_mat = p.pin;
        m = p.m;
        sig_t = T.xs4[(m * G + p.g) * 4];
        v = T.speed[p.g];
        // A3 distance to collision
        const U4 r = draw_block(p.pid, p.ectr, BLK_DCOL, seedb);
        double d_c = -mc_log(u52(r.x, r.y)) / sig_t;
        if (d_c < 0.0) d_c = 0.0;
        // A4 distance to surface: x, y, z, cylinder; strict < replaces
        double d_s = plane_dist(P.px, p.ix, p.x, p.ux);
        const double dsy = plane_dist(P.py, p.iy, p.y, p.uy);
        if (dsy < d_s) { d_s = dsy; surf = 1; }
        const double dsz = plane_dist(P.pz, p.iz, p.z, p.uz);
        if (dsz < d_s) { d_s = dsz; surf = 2; }
        if (pin_mat >= 0) {
          const double cx = 0.5 * (__ldg(P.px + p.ix) + __ldg(P.px + p.ix + 1));
          const double cy = 0.5 * (__ldg(P.py + p.iy) + __ldg(P.py + p.iy + 1));
          const double dcy = cyl_dist(p.x, p.y, p.ux, p.uy, cx, cy,
                                      __ldg(P.radius + (p.iz * P.ny + p.iy) * P.nx + p.ix), p.inside);
          if (dcy < d_s) { d_s = dcy; surf = 3; }
        }
        // A5 distance to census, event select (ties: collision, surface, census)
        double d_t = (t_k - p.t) * v;
        if (d_t < 0.0) d_t = 0.0;
        d = d_c; ev = 0;
        if (d_s < d) { d = d_s; ev = 1; }
        if (d_t < d) { d = d_t; ev = 2; }
      }
      // a flight counter at its 24-bit limit would repeat the random streams: the particle ends as lost (C.1)
      const bool worn = live && p.ectr == 0xFFFFFFu;
      if (worn) d = 0.0;

      // A6 tally march (warp-synchronous; never creates events, never draws)
      bool lost = false;
      bool generic = live;
      if (P.simple_tally) {
        // Tally planes bitwise equal to the lattice planes: when the coordinate lookup of
        // every axis lands in the particle's own cell and the next tally time edge is the
        // census time, each candidate crossing distance of the march equals the matching
        // event distance (same expression, same operands) and is therefore >= d: the march
        // is exactly one segment of length d in bin (jt, g, iz, iy, ix).  Any other case
        // (an ulp drift across a plane, intermediate time edges) takes the general march.
        long long bin = -1; double val = 0.0;
        if (live) {
          const double lx = __ldg(P.px + p.ix), hx = __ldg(P.px + p.ix + 1);
          const double ly = __ldg(P.py + p.iy), hy = __ldg(P.py + p.iy + 1);
          const double lz = __ldg(P.pz + p.iz), hz = __ldg(P.pz + p.iz + 1);
          const bool okx = (lx < p.x && p.x < hx) || (p.x == lx && (p.ux >= 0.0 || p.ix == 0)) ||
                           (p.x == hx && (p.ux < 0.0 || p.ix == P.nx - 1));
          const bool oky = (ly < p.y && p.y < hy) || (p.y == ly && (p.uy >= 0.0 || p.iy == 0)) ||
                           (p.y == hy && (p.uy < 0.0 || p.iy == P.ny - 1));
          const bool okz = (lz < p.z && p.z < hz) || (p.z == lz && (p.uz >= 0.0 || p.iz == 0)) ||
                           (p.z == hz && (p.uz < 0.0 || p.iz == P.nz - 1));
          if (okx && oky && okz) {
            // time bin: the one whose upper edge is this step's census time (found once per
            // launch); the particle is in it iff t_lo <= t < t_k
            if (jt_step >= 0 && p.t >= t_lo_step && p.t < t_k) {
              generic = false;
              if (d > 0.0) {
                bin = (long long)bin_t0 + (long long)(p.g * g_stride + (p.iz * P.tny + p.iy) * P.tnx + p.ix);
                val = p.w * d; ++c_segments;
              }
            }
          }
        }
        if (__any_sync(0xffffffffu, bin >= 0)) warp_tally_add(P.tally, bin, val, P.aggregate_tally != 0);
      }
      if (__any_sync(0xffffffffu, generic)) {
        int jx = 0, jy = 0, jz = 0, jt = 0;
        double sx = INF, sy = INF, sz = INF, st = INF, s_prev = 0.0;
        bool marching = generic;
        uint32_t nseg = 0;
        if (generic) {
          jx = find_interval_fast(P.tx, P.tnx, p.x, p.ux, P.hx);
          jy = find_interval_fast(P.ty, P.tny, p.y, p.uy, P.hy);
          jz = find_interval_fast(P.tz, P.tnz, p.z, p.uz, P.hz);
          jt = find_interval_fast(P.tt, P.tnt, p.t, 1.0, P.ht);
          sx = plane_dist(P.tx, jx, p.x, p.ux);
          sy = plane_dist(P.ty, jy, p.y, p.uy);
          sz = plane_dist(P.tz, jz, p.z, p.uz);
          st = (__ldg(P.tt + jt + 1) - p.t) * v; if (st < 0.0) st = 0.0;
        }
        for (;;) {
          long long bin = -1; double val = 0.0;
          if (marching) {
            int axis = 0; double s_min = sx;
            if (sy < s_min) { s_min = sy; axis = 1; }
            if (sz < s_min) { s_min = sz; axis = 2; }
            if (st < s_min) { s_min = st; axis = 3; }
            const bool cross = s_min < d;
            const double len = (cross ? s_min : d) - s_prev;
            if (len > 0.0) {
              bin = ((((long long)jt * G + p.g) * P.tnz + jz) * P.tny + jy) * P.tnx + jx;
              val = p.w * len; ++nseg;
            }
            if (cross) {
              if (axis == 0) { jx += (p.ux > 0.0) ? 1 : -1; if (jx < 0 || jx >= P.tnx) lost = true; else sx = plane_dist(P.tx, jx, p.x, p.ux); }
              else if (axis == 1) { jy += (p.uy > 0.0) ? 1 : -1; if (jy < 0 || jy >= P.tny) lost = true; else sy = plane_dist(P.ty, jy, p.y, p.uy); }
              else if (axis == 2) { jz += (p.uz > 0.0) ? 1 : -1; if (jz < 0 || jz >= P.tnz) lost = true; else sz = plane_dist(P.tz, jz, p.z, p.uz); }
              else { jt += 1; if (jt >= P.tnt) lost = true; else { st = (__ldg(P.tt + jt + 1) - p.t) * v; if (st < 0.0) st = 0.0; } }
              s_prev = s_min;
              if (lost) marching = false;
            } else marching = false;
          }
          if (!__any_sync(0xffffffffu, bin >= 0 || marching)) break;
          if (__any_sync(0xffffffffu, bin >= 0)) warp_tally_add(P.tally, bin, val, P.aggregate_tally != 0);
        }
        if (!lost) c_segments += nseg;
      }

      // move, snap, dispatch
      lost = lost || worn;
      if (live) {
        ++c_flights;
        if (lost) {
          ++c_lost; end_ev = END_LOST; end_pid = p.pid; end_ectr = p.ectr; live = false; outcome = 0;
        } else {
          p.x = fma(d, p.ux, p.x); p.y = fma(d, p.uy, p.y); p.z = fma(d, p.uz, p.z);
          p.t = p.t + d / v;
          if (ev == 2) {                                   // A11 census
            p.t = t_k; ++c_census; end_ev = END_CENSUS; end_pid = p.pid; end_ectr = p.ectr;
            ++p.ectr; live = false; outcome = last_step ? 0 : 3;
            if (WQ && outcome == 3) {                      // bank it now: the lane moves on to other work
              outcome = 0;
              uint32_t cs = slot;
              if (!slot_free) cs = nsp ? spare[--nsp] : atomicAdd(&ctl->bank_tail, 1u);
              slot_free = false;
              if (cs >= Q.capacity) atomicExch(&ctl->overflow, 1u);
              else {
                B.xy[cs] = make_double2(p.x, p.y); B.zt[cs] = make_double2(p.z, p.t);
                B.uxy[cs] = make_double2(p.ux, p.uy); B.uzw[cs] = make_double2(p.uz, p.w);
                B.idp[cs] = make_ulonglong2(p.pid, pack_state(p.ectr, p.g, p.ix, p.iy, p.iz, p.inside));
                Q.census[atomicAdd(&ctl->n_census, 1u)] = cs;
              }
            }
          } else if (ev == 1) {                            // A7 surface
            if (surf == 3) { p.inside ^= 1; p.m = p.inside ? p.pin : (int)__ldg(P.mat_outer + (p.iz * P.ny + p.iy) * P.nx + p.ix); ++c_cross; ++p.ectr; }
            else {
              const double u = surf == 0 ? p.ux : surf == 1 ? p.uy : p.uz;
              const bool up = u > 0.0;
              const int idx = surf == 0 ? p.ix : surf == 1 ? p.iy : p.iz;
              const int nax = surf == 0 ? P.nx : surf == 1 ? P.ny : P.nz;
              const double *pl = surf == 0 ? P.px : surf == 1 ? P.py : P.pz;
              const double edge = __ldg(pl + idx + (up ? 1 : 0));
              if (surf == 0) p.x = edge; else if (surf == 1) p.y = edge; else p.z = edge;
              const bool outer = up ? (idx == nax - 1) : (idx == 0);
              if (!outer) {
                const int ni = idx + (up ? 1 : -1);
                if (surf == 0) p.ix = ni; else if (surf == 1) p.iy = ni; else p.iz = ni;
                p.inside = 0; lane_material(P, p); ++c_cross; ++p.ectr;
              } else if (P.bc[2 * surf + (up ? 1 : 0)] == 1) {
                if (surf == 0) p.ux = -p.ux; else if (surf == 1) p.uy = -p.uy; else p.uz = -p.uz;
                dir_dirty = true; ++c_refl; ++p.ectr;
              } else { ++c_leak; end_ev = END_LEAK; end_pid = p.pid; end_ectr = p.ectr; live = false; outcome = 0; }
            }
          } else if (!FUSE) {                              // collision: queued for k_collide
            live = false; outcome = 2;
          } else {                                         // A8-A10 in place
            const double *xs = T.xs4 + (m * G + p.g) * 4;
            const double ssr = xs[1], sf = xs[2], nu = xs[3];
            ++c_coll;
            const U4 r = draw_block(p.pid, p.ectr, BLK_REACT, seedb);
            const double a = u52(r.x, r.y) * sig_t;
            if (a < ssr) {
              ++c_scat;
              p.g = sample_cdf(T.cdf_s + (m * G + p.g) * G, G, u52(r.z, r.w));
              const U4 rd = draw_block(p.pid, p.ectr, BLK_SCAT_DIR, seedb);
              isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), p.ux, p.uy, p.uz);
              dir_dirty = true; ++p.ectr;
            } else if (a < ssr + sf) {
              ++c_fis; end_ev = END_FISSION; end_pid = p.pid; end_ectr = p.ectr;
              const U4 rn = draw_block(p.pid, p.ectr, BLK_FIS_N, seedb);
              uint32_t nch = (uint32_t)(int)(nu + u52(rn.x, rn.y));
              c_sec += nch;
              if (nch == 0) { live = false; outcome = 0; }
              else {
                const uint64_t ppid = p.pid; const uint32_t pectr = p.ectr;
                for (uint32_t j = nch; j-- > 0;) {            // child 0 last: the lane adopts it
                  const U4 rc = draw_block(ppid, pectr, BLK_CHILD + j, seedb);
                  const uint64_t cpid = (1ull << 63) | ((((uint64_t)rc.x << 32) | (uint64_t)rc.y) >> 1);
                  const U4 rg = draw_block(cpid, 0, BLK_SRC_ZG, seedb);
                  const int cg = sample_cdf(T.cdf_chi + m * G, G, u52(rg.z, rg.w));
                  const U4 rd = draw_block(cpid, 0, BLK_SRC_DIR, seedb);
                  double cux, cuy, cuz;
                  isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), cux, cuy, cuz);
                  if (j) {                                    // banked for the next launch
                    const uint32_t cs = (WQ && nsp) ? spare[--nsp] : atomicAdd(&ctl->bank_tail, 1u);
                    if (cs >= Q.capacity) { atomicExch(&ctl->overflow, 1u); continue; }
                    B.xy[cs] = make_double2(p.x, p.y); B.zt[cs] = make_double2(p.z, p.t);
                    B.uxy[cs] = make_double2(cux, cuy); B.uzw[cs] = make_double2(cuz, p.w);
                    B.idp[cs] = make_ulonglong2(cpid, pack_state(0, cg, p.ix, p.iy, p.iz, p.inside));
                    if (WQ) {                                 // publish to the work queue
                      const uint32_t pos = atomicAdd(&ctl->wq_tail, 1u);
                      if (pos - n < Q.capacity) {
                        __threadfence();
                        atomicAdd(&ctl->wq_pending, 1u);
                        *(volatile uint32_t *)(q_out + (pos - n)) = cs + 1u;
                      } else {
                        // the published region is full (a launch publishes without bound in a multiplying medium while
                        // bank slots are recycled): the child waits in the collision list, unused in this mode, which
                        // k_tail_spill turns into the active queue of the next launch
                        Q.coll[atomicAdd(&ctl->n_coll, 1u)] = cs;
                      }
                    } else q_out[atomicAdd(&ctl->n_next, 1u)] = cs;
                  } else {
                    p.pid = cpid; p.ectr = 0; p.g = cg; p.ux = cux; p.uy = cuy; p.uz = cuz;
                    dir_dirty = true;
                  }
                }
              }
            } else { ++c_capt; end_ev = END_CAPTURE; end_pid = p.pid; end_ectr = p.ectr; live = false; outcome = 0; }
          }
          if (live && ++nfl >= max_flights) { live = false; outcome = 1; }
        }
      }
      if (end_ev >= 0) fp += end_hash(end_pid, end_ectr, end_ev);      // one place for every kind of end
      if (REFILL) {                       // hand in the particles that left the loop in this round
        const bool fin = was_live && !live;
        if (fin && outcome != 0) {
          B.xy[slot] = make_double2(p.x, p.y);
          B.zt[slot] = make_double2(p.z, p.t);
          if (dir_dirty) { B.uxy[slot] = make_double2(p.ux, p.uy); B.uzw[slot] = make_double2(p.uz, p.w); }
          B.idp[slot] = make_ulonglong2(p.pid, pack_state(p.ectr, p.g, p.ix, p.iy, p.iz, p.inside));
        }
        const unsigned mc = __ballot_sync(0xffffffffu, fin && outcome == 2);
        const unsigned ms = __ballot_sync(0xffffffffu, fin && outcome == 3);
        if (fin && outcome == 2) s_stage[warp_id][0][n_st_coll + __popc(mc & lt_mask)] = slot;
        if (fin && outcome == 3) s_stage[warp_id][1][n_st_cens + __popc(ms & lt_mask)] = slot;
        n_st_coll += __popc(mc); n_st_cens += __popc(ms);
        __syncwarp();
        if (n_st_coll >= (uint32_t)STAGE_FLUSH) { stage_flush(s_stage[warp_id][0], n_st_coll, &ctl->n_coll, Q.coll); n_st_coll = 0; }
        if (n_st_cens >= (uint32_t)STAGE_FLUSH) { stage_flush(s_stage[warp_id][1], n_st_cens, &ctl->n_census, Q.census); n_st_cens = 0; }
      }
      if (WQ && was_live && !live) {                                   // this particle is finished
        if (slot_free && nsp < N_SPARE) spare[nsp++] = slot;
        atomicSub(&ctl->wq_pending, 1u);
      }
    }

    if (REFILL) {
      stage_flush(s_stage[warp_id][0], n_st_coll, &ctl->n_coll, Q.coll);
      stage_flush(s_stage[warp_id][1], n_st_cens, &ctl->n_census, Q.census);
      outcome = 0;
    }
    if (outcome != 0) {
      B.xy[slot] = make_double2(p.x, p.y);
      B.zt[slot] = make_double2(p.z, p.t);
      if (dir_dirty) { B.uxy[slot] = make_double2(p.ux, p.uy); B.uzw[slot] = make_double2(p.uz, p.w); }
      B.idp[slot] = make_ulonglong2(p.pid, pack_state(p.ectr, p.g, p.ix, p.iy, p.iz, p.inside));
    }

    // A13 compaction into the per-event queues (the refill kernel has appended already)
    if (!REFILL) {
      uint32_t pos = block_reserve1(outcome == 1, &ctl->n_next, s_w);
      if (outcome == 1) q_out[pos] = slot;
      if (!FUSE) {
        pos = block_reserve1(outcome == 2, &ctl->n_coll, s_w);
        if (outcome == 2) Q.coll[pos] = slot;
      }
      if (!last_step) {
        pos = block_reserve1(outcome == 3, &ctl->n_census, s_w);
        if (outcome == 3) Q.census[pos] = slot;
      }
    }
  }

  warp_count(s_cnt, K_FLIGHTS, c_flights);
  warp_count(s_cnt, K_SEGMENTS, c_segments);
  warp_count(s_cnt, K_CROSSINGS, c_cross);
  warp_count(s_cnt, K_REFLECTIONS, c_refl);
  warp_count(s_cnt, K_LEAKS, c_leak);
  warp_count(s_cnt, K_CENSUS, c_census);
  warp_count(s_cnt, K_LOST, c_lost);
  if (FUSE) {
    warp_count(s_cnt, K_COLLISIONS, c_coll);
    warp_count(s_cnt, K_SCATTERS, c_scat);
    warp_count(s_cnt, K_CAPTURES, c_capt);
    warp_count(s_cnt, K_FISSIONS, c_fis);
    warp_count(s_cnt, K_SECONDARIES, c_sec);
  }
  warp_count64(s_cnt, K_FINGERPRINT, fp);
  flush_counts(s_cnt, ctl->cnt);
}


// ---- A8-A10: collisions: reaction select, scatter with group transfer, fission
// with secondary banking (atomic append), capture.
__global__ void __launch_bounds__(BS, MB_COLLIDE) k_collide(DevProblem P, TableLayout L, int use_smem, Bank B,
                                                Ctl *ctl, Queues Q)
{
  extern __shared__ double smem[];
  __shared__ uint32_t s_w[NWARP + 1];
  __shared__ uint32_t s_free[BS];
  __shared__ uint32_t s_base, s_qbase;
  __shared__ unsigned long long s_cnt[N_CNT];
  const Tables T = stage_tables(P, L, smem, use_smem);
  if (threadIdx.x < N_CNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const uint32_t n = ctl->n_coll;
  uint32_t *__restrict__ q_out = Q.q[ctl->parity ^ 1u];
  const unsigned long long seedb = ctl->seedb;
  const int G = P.G;
  uint32_t c_coll = 0, c_scat = 0, c_capt = 0, c_fis = 0, c_sec = 0;
  unsigned long long fp = 0ull;

  for (uint32_t base = blockIdx.x * BS; base < n; base += gridDim.x * BS) {
    const uint32_t i = base + threadIdx.x;
    const bool valid = i < n;
    uint32_t slot = 0, n_out = 0, n_new = 0;
    uint64_t pid = 0, pk = 0;
    uint32_t ectr = 0;
    int m = 0, kind = 0;            // kind: 0 capture, 1 scatter, 2 fission
    double w = 0.0;
    if (valid) {
      slot = Q.coll[i];
      const ulonglong2 id = B.idp[slot];
      const double2 e2 = B.uzw[slot];             // issued with the id load: w is needed by every outcome but capture
      w = e2.y;
      pid = id.x; pk = id.y; ectr = pk_ectr(pk);
      const int g = pk_g(pk);
      const int cell = (pk_iz(pk) * P.ny + pk_iy(pk)) * P.nx + pk_ix(pk);
      m = pk_inside(pk) ? (int)P.mat_inner[cell] : (int)P.mat_outer[cell];
      const double *xs = T.xs4 + (m * G + g) * 4;
      const double sig_t = xs[0], ssr = xs[1], sf = xs[2], nu = xs[3];
      ++c_coll;
      const U4 r = draw_block(pid, ectr, BLK_REACT, seedb);
      const double a = u52(r.x, r.y) * sig_t;
      if (a < ssr) {
        kind = 1; n_out = 1; ++c_scat;
        const int g2 = sample_cdf(T.cdf_s + (m * G + g) * G, G, u52(r.z, r.w));
        const U4 rd = draw_block(pid, ectr, BLK_SCAT_DIR, seedb);
        double ux, uy, uz;
        isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
        B.uxy[slot] = make_double2(ux, uy);
        B.uzw[slot] = make_double2(uz, w);
        pk = (pk & ~(0xFFull << 32)) | ((uint64_t)(uint32_t)g2 << 32);
        pk = (pk & 0x000000FFFFFFFFFFull) | ((uint64_t)(ectr + 1u) << 40);
        B.idp[slot] = make_ulonglong2(pid, pk);
      } else if (a < ssr + sf) {
        kind = 2; ++c_fis;
        const U4 rn = draw_block(pid, ectr, BLK_FIS_N, seedb);
        n_out = (uint32_t)(int)(nu + u52(rn.x, rn.y));
        c_sec += n_out;
        n_new = n_out > 0 ? n_out - 1 : 0;
        fp += end_hash(pid, ectr, END_FISSION);
      } else { ++c_capt; fp += end_hash(pid, ectr, END_CAPTURE); }
    }
    // A10 secondary banking: extra children first take the slots of the particles this
    // block has just seen captured, then fresh slots at the bank tail (one atomic per block)
    // (one block scan over the packed triple give | need << 10 | out << 21)
    const uint32_t give = (valid && kind == 0) ? 1u : 0u;
    uint32_t tot;
    const uint32_t pre = block_scan_total(give | (n_new << 10) | (n_out << 21), s_w, tot);
    const uint32_t gpos = pre & 0x3FFu, npos = (pre >> 10) & 0x7FFu;
    const uint32_t tot_give = tot & 0x3FFu, tot_need = (tot >> 10) & 0x7FFu, tot_out = tot >> 21;
    if (give) s_free[gpos] = slot;
    if (threadIdx.x == 0) {
      const uint32_t fresh = tot_need > tot_give ? tot_need - tot_give : 0u;
      s_base = fresh ? atomicAdd(&ctl->bank_tail, fresh) : 0u;
      if (fresh && s_base + fresh > Q.capacity) { atomicExch(&ctl->overflow, 1u); s_base = 0xFFFFFFFFu; }
      s_qbase = tot_out ? atomicAdd(&ctl->n_next, tot_out) : 0u;
    }
    __syncthreads();
    const uint32_t qpos = s_qbase + (pre >> 21);
    if (s_base == 0xFFFFFFFFu && n_new) { n_out -= n_new; n_new = 0; }     // bank full: run invalid (queue holes are never read)
    if (kind == 1) q_out[qpos] = slot;
    else if (kind == 2 && n_out) {
      const double2 a2 = B.xy[slot], b2 = B.zt[slot];
      for (uint32_t j = 0; j < n_out; ++j) {
        const U4 rc = draw_block(pid, ectr, BLK_CHILD + j, seedb);
        const uint64_t cpid = (1ull << 63) | ((((uint64_t)rc.x << 32) | (uint64_t)rc.y) >> 1);
        const U4 rg = draw_block(cpid, 0, BLK_SRC_ZG, seedb);
        const int cg = sample_cdf(T.cdf_chi + m * G, G, u52(rg.z, rg.w));
        const U4 rd = draw_block(cpid, 0, BLK_SRC_DIR, seedb);
        double ux, uy, uz;
        isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
        const uint32_t fi = npos + (j - 1);
        const uint32_t cs = (j == 0) ? slot : (fi < tot_give ? s_free[fi] : s_base + (fi - tot_give));
        if (j) { B.xy[cs] = a2; B.zt[cs] = b2; }
        B.uxy[cs] = make_double2(ux, uy);
        B.uzw[cs] = make_double2(uz, w);
        uint64_t cpk = (pk & 0x00000000FFFFFFFFull) | ((uint64_t)(uint32_t)cg << 32);
        B.idp[cs] = make_ulonglong2(cpid, cpk);
        q_out[qpos + j] = cs;
      }
    }
  }
  warp_count(s_cnt, K_COLLISIONS, c_coll);
  warp_count(s_cnt, K_SCATTERS, c_scat);
  warp_count(s_cnt, K_CAPTURES, c_capt);
  warp_count(s_cnt, K_FISSIONS, c_fis);
  warp_count(s_cnt, K_SECONDARIES, c_sec);
  warp_count64(s_cnt, K_FINGERPRINT, fp);
  flush_counts(s_cnt, ctl->cnt);
}

// ---- work queue of the tail kernel: tickets 0..n-1 are the active queue
__global__ void k_tail_begin(Ctl *ctl)
{
  ctl->wq_head = 0u; ctl->wq_tail = ctl->n_active; ctl->wq_pending = ctl->n_active;
}

// children the tail kernel could not publish (Q.coll) become the next queue; the launch that follows takes them
__global__ void __launch_bounds__(BS) k_tail_spill(Ctl *ctl, Queues Q)
{
  const uint32_t n = ctl->n_coll;
  uint32_t *__restrict__ q_out = Q.q[ctl->parity ^ 1u];
  for (uint32_t i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS) q_out[i] = Q.coll[i];
  if (blockIdx.x == 0 && threadIdx.x == 0) ctl->n_next = n;
}

// ---- end of one event-loop iteration: the next queue becomes the active one
__global__ void k_flip(Ctl *ctl, uint32_t *host_n_active)
{
  ctl->n_active = ctl->n_next;
  ctl->n_next = 0u; ctl->n_coll = 0u; ctl->fetch = 0u;
  ctl->parity ^= 1u;
  ctl->iter += 1u;
  if (host_n_active) { host_n_active[0] = ctl->n_active; host_n_active[1] = ctl->n_census; host_n_active[2] = ctl->overflow; host_n_active[3] = ctl->bank_tail;
    host_n_active[4] = (uint32_t)ctl->cnt[K_FLIGHTS]; host_n_active[5] = (uint32_t)(ctl->cnt[K_FLIGHTS] >> 32); }
}

}  // namespace mcdc
