// mcdc_pool.cu — one census step of the history loop as ONE persistent launch
// (SURVEY §8(a) rows A0, A2-A11, A13).  Definitions: DESIGN.md §3; design: DESIGN.md §6.
//
// Every warp keeps a pool of PW particles in shared memory (80-byte records + material) and
// per-event lists of pool slots: flight-ready, collision-ready, unborn fission children, waiting
// for the census write-out, free.  A round takes up to 32 slots of ONE list, so all lanes of the warp run
// the same event code (the divergence between flying and colliding particles that the paper
// hands to an asynchronous scheduler, is removed by construction).  Particles
// enter the pool from the dense active bank (coalesced 128-bit loads, ranges reserved with one
// atomic per warp and chunk) and leave it either dead or through the census write-out (32
// records at a time, one atomic, coalesced 128-bit stores into the other bank).  Between
// entry and exit a particle never touches HBM; only tally adds and the material map do.
// Fission children take free pool slots (a fission whose children do not fit is retried later:
// the counter-based RNG makes the retry identical); only when a pool is full of such parents are
// children appended to the active bank behind the range being processed, and the host relaunches
// over that range.  Terminal events are hashed into the fingerprint 32 at a time from a ring.
#include "mcdc_kernels.cuh"

namespace mcdc {

#ifndef POOL_PW
#define POOL_PW 96                 // pool slots per warp (<= 256: lists are bytes)
#endif
#ifndef POOL_RESERVE
#define POOL_RESERVE 16            // pool slots kept free for fission children when particles are dealt in
#endif
#ifndef MB_POOL
#define MB_POOL 2
#endif
#ifndef POOL_NT
#define POOL_NT 256                // threads per block
#endif
constexpr int PW = POOL_PW;
constexpr int POOL_THREADS = POOL_NT;
constexpr int POOL_WARPS = POOL_THREADS / 32;
constexpr int HRING = 64;                              // terminal events waiting for their fingerprint hash
constexpr int POOL_BYTES = PW * (80 + 4) + 5 * PW + HRING * 12;   // records, material, five byte lists, hash ring
static_assert(POOL_BYTES % 16 == 0, "pool alignment");

static __host__ __device__ __forceinline__ size_t pool_table_bytes(const TableLayout &L, int use_smem)
{
  return use_smem ? (((size_t)L.total * 8 + 15) & ~(size_t)15) : 0;
}

// pool record <-> registers
static __device__ __forceinline__ int mat_pack(int m, int pin) { return (m & 0xFF) | ((pin + 1) << 8); }

__global__ void __launch_bounds__(POOL_THREADS, MB_POOL)
k_pool(DevProblem P, TableLayout L, int use_smem, Bank Bin, Bank Bout, Ctl *ctl, Queues Q,
       int max_flights, uint32_t fetch_chunk)
{
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ unsigned long long s_cnt[N_CNT];
  const Tables T = stage_tables(P, L, (double *)smem_raw, use_smem);
  if (threadIdx.x < N_CNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  unsigned char *pool = smem_raw + pool_table_bytes(L, use_smem) + (size_t)wid * POOL_BYTES;
  double2 *const s_xy = (double2 *)pool;
  double2 *const s_zt = s_xy + PW;
  double2 *const s_uxy = s_zt + PW;
  double2 *const s_uzw = s_uxy + PW;
  ulonglong2 *const s_idp = (ulonglong2 *)(s_uzw + PW);
  unsigned long long *const h_pid = (unsigned long long *)(s_idp + PW);   // hash ring: id, (ectr | event << 24)
  int *const s_mat = (int *)(h_pid + HRING);        // material | (pin + 1) << 8 | child index << 16
  uint32_t *const h_ce = (uint32_t *)(s_mat + PW);
  uint8_t *const l_f = (uint8_t *)(h_ce + HRING);   // flight-ready
  uint8_t *const l_c = l_f + PW;                    // collision-ready
  uint8_t *const l_b = l_c + PW;                    // fission children waiting to be born
  uint8_t *const l_z = l_b + PW;                    // waiting for the census write-out
  uint8_t *const l_free = l_z + PW;
  for (int i = lane; i < PW; i += 32) l_free[i] = (uint8_t)i;
  __syncwarp();
  uint32_t nF = 0, nC = 0, nB = 0, nZ = 0, nFree = PW, nH = 0;     // warp-uniform list lengths
  bool blocked = false;                             // the last collision round had to put fissions back

  const uint32_t n_end = ctl->n_active;             // active bank range [fetch, n_end)
  const uint32_t spill_limit = ctl->spill_limit;
  const double t_k = ctl->t_k;
  const unsigned long long seedb = ctl->seedb;
  const bool last_step = ctl->last_step != 0u;
  const double INF = d_inf();
  const int G = P.G;
  // simple-tally path: time bin of this census step (see k_flight)
  int jt_step = -1;
  if (P.simple_tally) {
    int lo = 0, hi = P.tnt;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(P.tt + mid) < t_k) lo = mid; else hi = mid; }
    if (__ldg(P.tt + lo + 1) == t_k) jt_step = lo;
    else if (__ldg(P.tt + 1) == t_k) jt_step = 0;
  }
  const double t_lo_step = jt_step >= 0 ? __ldg(P.tt + jt_step) : 0.0;
  const int g_stride = P.tnz * P.tny * P.tnx;
  if (!((long long)g_stride * G < (1ll << 30))) jt_step = -1;
  const long long bin_t0 = (long long)(jt_step >= 0 ? jt_step : 0) * G * g_stride;

  uint32_t c_flights = 0, c_segments = 0, c_cross = 0, c_refl = 0, c_leak = 0, c_census = 0, c_lost = 0;
  uint32_t c_coll = 0, c_scat = 0, c_capt = 0, c_fis = 0, c_sec = 0;
  unsigned long long fp = 0ull;

  uint32_t rng_next = 0, rng_end = 0, round = 0;
  bool exhausted = false;

  // terminal events wait in a ring and are hashed into the fingerprint 32 at a time
  auto ring_push = [&](bool has, uint64_t pid, uint32_t ectr, int ev) {
    const unsigned b = __ballot_sync(0xffffffffu, has);
    if (b == 0u) return;
    if (has) { const uint32_t k = nH + __popc(b & lt_mask); h_pid[k] = pid; h_ce[k] = ectr | ((uint32_t)ev << 24); }
    nH += __popc(b);
    __syncwarp();
    if (nH >= 32u) {
      nH -= 32u;
      fp += end_hash(h_pid[nH + lane], h_ce[nH + lane] & 0xFFFFFFu, (int)(h_ce[nH + lane] >> 24));
      __syncwarp();
    }
  };

  for (;;) {
    // ---- entry: deal reserved entries of the active bank to free pool slots ----
    if (nF < 32u && nFree > (uint32_t)POOL_RESERVE && !exhausted) {
      if (rng_next == rng_end) {
        uint32_t b = 0;
        if (lane == 0) b = atomicAdd(&ctl->fetch, fetch_chunk);
        b = __shfl_sync(0xffffffffu, b, 0);
        rng_next = min(b, n_end); rng_end = min(b + fetch_chunk, n_end);
        if (rng_next == rng_end) exhausted = true;
      }
      if (!exhausted) {
        const uint32_t cnt = min(min(nFree - (uint32_t)POOL_RESERVE, 32u), rng_end - rng_next);
        if ((uint32_t)lane < cnt) {
          const uint32_t slot = l_free[nFree - 1u - lane];
          const uint32_t i = rng_next + lane;
          const double2 a = Bin.xy[i], b2 = Bin.zt[i], c2 = Bin.uxy[i], e2 = Bin.uzw[i];
          const ulonglong2 id = Bin.idp[i];
          s_xy[slot] = a; s_zt[slot] = b2; s_uxy[slot] = c2; s_uzw[slot] = e2; s_idp[slot] = id;
          const int cell = (pk_iz(id.y) * P.ny + pk_iy(id.y)) * P.nx + pk_ix(id.y);
          const int pin = P.has_pins ? (int)__ldg(P.mat_inner + cell) : -1;
          const int m = pk_inside(id.y) ? pin : (int)__ldg(P.mat_outer + cell);
          s_mat[slot] = mat_pack(m, pin);
          l_f[nF + lane] = (uint8_t)slot;
        }
        nFree -= cnt; nF += cnt; rng_next += cnt;
        __syncwarp();
      }
    }
    // ---- exit: census write-out, 32 records per atomic ----
    if (nZ >= 32u || (nZ > 0u && ((nF == 0u && nC == 0u && nB == 0u) || blocked))) {
      const uint32_t cnt = min(nZ, 32u);
      uint32_t pos = 0;
      if (lane == 0) pos = atomicAdd(&ctl->n_census, cnt);
      pos = __shfl_sync(0xffffffffu, pos, 0);
      const bool room = pos + cnt <= Q.capacity;
      if (!room && lane == 0) atomicExch(&ctl->overflow, 1u);
      if ((uint32_t)lane < cnt) {
        const uint32_t slot = l_z[nZ - 1u - lane];
        if (room) {
          const uint32_t o = pos + lane;
          Bout.xy[o] = s_xy[slot]; Bout.zt[o] = s_zt[slot]; Bout.uxy[o] = s_uxy[slot];
          Bout.uzw[o] = s_uzw[slot]; Bout.idp[o] = s_idp[slot];
          Q.census[o] = o;
        }
        l_free[nFree + lane] = (uint8_t)slot;
      }
      nZ -= cnt; nFree += cnt;
      __syncwarp();
    }
    if (nF == 0u && nC == 0u && nB == 0u) {
      if (exhausted && nZ == 0u) break;
      continue;
    }
    if ((round++ & 63u) == 63u) {                                                  // run is invalid: stop
      uint32_t ov = 0;
      if (lane == 0) ov = ld_volatile_u32(&ctl->overflow);
      if (__shfl_sync(0xffffffffu, ov, 0) != 0u) break;
    }

    // one event kind per round: a full warp of one kind if there is one, else the longest list
    // (after a collision round that had to put fissions back, anything else goes first)
    int pick;                                         // 0 flight, 1 collision, 2 birth
    if (nB >= 32u) pick = 2;
    else if (nC >= 32u && !blocked) pick = 1;
    else if (nF >= 32u) pick = 0;
    else if (blocked && (nB | nF)) pick = nB >= nF ? 2 : 0;
    else pick = (nB >= nC && nB >= nF) ? 2 : (nC >= nF ? 1 : 0);

    if (pick == 0) {
      blocked = false;
      // ================= flight round (A3-A7, A11) =================
      const uint32_t cnt = min(nF, 32u);
      const bool active = (uint32_t)lane < cnt;
      const uint32_t slot = active ? l_f[nF - 1u - lane] : 0u;
      nF -= cnt;
      Lane p;
      p.x = p.y = p.z = p.t = 0.0; p.ux = 1.0; p.uy = p.uz = 0.0; p.w = 0.0;
      p.pid = 0; p.ectr = 0; p.g = 0; p.ix = p.iy = p.iz = 0; p.inside = 0; p.m = 0; p.pin = -1;
      if (active) {
        const double2 a = s_xy[slot], b2 = s_zt[slot], c2 = s_uxy[slot], e2 = s_uzw[slot];
        const ulonglong2 id = s_idp[slot];
        const int mm = s_mat[slot];
        p.x = a.x; p.y = a.y; p.z = b2.x; p.t = b2.y; p.ux = c2.x; p.uy = c2.y; p.uz = e2.x; p.w = e2.y;
        p.pid = id.x;
        p.ectr = pk_ectr(id.y); p.g = pk_g(id.y); p.ix = pk_ix(id.y); p.iy = pk_iy(id.y);
        p.iz = pk_iz(id.y); p.inside = pk_inside(id.y);
        p.m = mm & 0xFF; p.pin = (mm >> 8) - 1;
      }
      bool live = active, dir_dirty = false;
      int outcome = 0;                  // 0 dead, 1 flight-ready, 2 collision, 3 census bank
      int nfl = 0;
      do {
        double d = 0.0, v = 1.0;
        int ev = 0, surf = 0;
        int end_ev = -1; uint64_t end_pid = 0; uint32_t end_ectr = 0;
        if (live) {
          const double sig_t = T.xs4[(p.m * G + p.g) * 4];
          v = T.speed[p.g];
          const U4 r = draw_block(p.pid, p.ectr, BLK_DCOL, seedb);
          double d_c = -mc_log(u52(r.x, r.y)) / sig_t;
          if (d_c < 0.0) d_c = 0.0;
          double d_s = plane_dist(P.px, p.ix, p.x, p.ux);
          const double dsy = plane_dist(P.py, p.iy, p.y, p.uy);
          if (dsy < d_s) { d_s = dsy; surf = 1; }
          const double dsz = plane_dist(P.pz, p.iz, p.z, p.uz);
          if (dsz < d_s) { d_s = dsz; surf = 2; }
          if (p.pin >= 0) {
            const double cx = 0.5 * (__ldg(P.px + p.ix) + __ldg(P.px + p.ix + 1));
            const double cy = 0.5 * (__ldg(P.py + p.iy) + __ldg(P.py + p.iy + 1));
            const double dcy = cyl_dist(p.x, p.y, p.ux, p.uy, cx, cy,
                                        __ldg(P.radius + (p.iz * P.ny + p.iy) * P.nx + p.ix), p.inside);
            if (dcy < d_s) { d_s = dcy; surf = 3; }
          }
          double d_t = (t_k - p.t) * v;
          if (d_t < 0.0) d_t = 0.0;
          d = d_c; ev = 0;
          if (d_s < d) { d = d_s; ev = 1; }
          if (d_t < d) { d = d_t; ev = 2; }
        }
        // A6 tally march (warp-synchronous; same two paths as k_flight)
        bool lost = false;
        bool generic = live;
        if (P.simple_tally) {
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
            if (okx && oky && okz && jt_step >= 0 && p.t >= t_lo_step && p.t < t_k) {
              generic = false;
              if (d > 0.0) {
                bin = (long long)bin_t0 + (long long)(p.g * g_stride + (p.iz * P.tny + p.iy) * P.tnx + p.ix);
                val = p.w * d; ++c_segments;
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
            } else if (ev == 1) {                            // A7 surface
              outcome = 1;
              if (surf == 3) {
                p.inside ^= 1;
                p.m = p.inside ? p.pin : (int)__ldg(P.mat_outer + (p.iz * P.ny + p.iy) * P.nx + p.ix);
                ++c_cross; ++p.ectr;
              } else {
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
            } else { live = false; outcome = 2; }            // collision: next round of that kind
          }
        }
        ring_push(end_ev >= 0, end_pid, end_ectr, end_ev);
      } while (++nfl < max_flights && __any_sync(0xffffffffu, live));
      // back to the pool, onto the list of the next event
      if (active && outcome != 0) {
        s_xy[slot] = make_double2(p.x, p.y);
        s_zt[slot] = make_double2(p.z, p.t);
        if (dir_dirty) { s_uxy[slot] = make_double2(p.ux, p.uy); s_uzw[slot] = make_double2(p.uz, p.w); }
        s_idp[slot] = make_ulonglong2(p.pid, pack_state(p.ectr, p.g, p.ix, p.iy, p.iz, p.inside));
        s_mat[slot] = mat_pack(p.m, p.pin);
      }
      const unsigned b1 = __ballot_sync(0xffffffffu, active && outcome == 1);
      const unsigned b2 = __ballot_sync(0xffffffffu, active && outcome == 2);
      const unsigned b3 = __ballot_sync(0xffffffffu, active && outcome == 3);
      const unsigned b0 = __ballot_sync(0xffffffffu, active && outcome == 0);
      if (active) {
        if (outcome == 1) l_f[nF + __popc(b1 & lt_mask)] = (uint8_t)slot;
        else if (outcome == 2) l_c[nC + __popc(b2 & lt_mask)] = (uint8_t)slot;
        else if (outcome == 3) l_z[nZ + __popc(b3 & lt_mask)] = (uint8_t)slot;
        else l_free[nFree + __popc(b0 & lt_mask)] = (uint8_t)slot;
      }
      nF += __popc(b1); nC += __popc(b2); nZ += __popc(b3); nFree += __popc(b0);
      __syncwarp();
    } else if (pick == 1) {
      // ================= collision round (A8-A10) =================
      const uint32_t cnt = min(nC, 32u);
      const bool active = (uint32_t)lane < cnt;
      const uint32_t slot = active ? l_c[nC - 1u - lane] : 0u;
      nC -= cnt;
      uint32_t n_out = 0, n_new = 0, ectr = 0;
      uint64_t pid = 0, pk = 0;
      int m = 0, kind = 0;              // kind: 0 capture, 1 scatter, 2 fission, 3 fission put back
      double w = 0.0;
      if (active) {
        const ulonglong2 id = s_idp[slot];
        w = s_uzw[slot].y;
        pid = id.x; pk = id.y; ectr = pk_ectr(pk);
        const int g = pk_g(pk);
        m = s_mat[slot] & 0xFF;
        const double *xs = T.xs4 + (m * G + g) * 4;
        const double sig_t = xs[0], ssr = xs[1], sf = xs[2], nu = xs[3];
        const U4 r = draw_block(pid, ectr, BLK_REACT, seedb);
        const double a = u52(r.x, r.y) * sig_t;
        if (a < ssr) {
          kind = 1;
          const int g2 = sample_cdf(T.cdf_s + (m * G + g) * G, G, u52(r.z, r.w));
          const U4 rd = draw_block(pid, ectr, BLK_SCAT_DIR, seedb);
          double ux, uy, uz;
          isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
          s_uxy[slot] = make_double2(ux, uy);
          s_uzw[slot] = make_double2(uz, w);
          pk = (pk & ~(0xFFull << 32)) | ((uint64_t)(uint32_t)g2 << 32);
          pk = (pk & 0x000000FFFFFFFFFFull) | ((uint64_t)(ectr + 1u) << 40);
          s_idp[slot] = make_ulonglong2(pid, pk);
        } else if (a < ssr + sf) {
          kind = 2;
          const U4 rn = draw_block(pid, ectr, BLK_FIS_N, seedb);
          n_out = (uint32_t)(int)(nu + u52(rn.x, rn.y));
          n_new = n_out > 0 ? n_out - 1 : 0;
        }
      }
      // slots of particles that ended are free before the children ask for room
      const bool dies = active && (kind == 0 || (kind == 2 && n_out == 0u));
      const unsigned bd = __ballot_sync(0xffffffffu, dies);
      if (dies) l_free[nFree + __popc(bd & lt_mask)] = (uint8_t)slot;
      nFree += __popc(bd);
      blocked = false;
      if (__ballot_sync(0xffffffffu, n_new > 0u)) {          // A10 secondary banking
        __syncwarp();
        uint32_t incl = n_new;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
          if (lane >= o) incl += t;
        }
        bool defer = n_new > 0u && incl > nFree;             // the family does not fit (in lane order)
        const unsigned bdef = __ballot_sync(0xffffffffu, defer);
        if (bdef) {
          const bool stuck = bdef == __ballot_sync(0xffffffffu, active) && nF == 0u && nB == 0u;
          if (!stuck) {
            // put back: the same collision is drawn again later from the same counters
            if (defer) { kind = 3; l_c[nC + __popc(bdef & lt_mask)] = (uint8_t)slot; n_new = 0; }
            nC += __popc(bdef); blocked = true;
          } else {
            // a pool full of fission parents: their further children go behind the active range
            uint32_t isp = defer ? n_new : 0u;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
              const uint32_t t = __shfl_up_sync(0xffffffffu, isp, o);
              if (lane >= o) isp += t;
            }
            const uint32_t n_spill = __shfl_sync(0xffffffffu, isp, 31);
            uint32_t spill_base = 0;
            if (lane == 0) spill_base = atomicAdd(&ctl->bank_tail, n_spill);
            spill_base = __shfl_sync(0xffffffffu, spill_base, 0);
            if (spill_base + n_spill > spill_limit) { if (lane == 0) atomicExch(&ctl->overflow, 1u); spill_base = 0xFFFFFFFFu; }
            if (defer && spill_base != 0xFFFFFFFFu) {
              const double2 a2 = s_xy[slot], b2 = s_zt[slot];
              for (uint32_t j = 1; j < n_out; ++j) {
                const U4 rc = draw_block(pid, ectr, BLK_CHILD + j, seedb);
                const uint64_t cpid = (1ull << 63) | ((((uint64_t)rc.x << 32) | (uint64_t)rc.y) >> 1);
                const U4 rg = draw_block(cpid, 0, BLK_SRC_ZG, seedb);
                const int cg = sample_cdf(T.cdf_chi + m * G, G, u52(rg.z, rg.w));
                const U4 rd = draw_block(cpid, 0, BLK_SRC_DIR, seedb);
                double ux, uy, uz;
                isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
                const uint32_t o = spill_base + (isp - n_new) + (j - 1u);
                Bin.xy[o] = a2; Bin.zt[o] = b2;
                Bin.uxy[o] = make_double2(ux, uy);
                Bin.uzw[o] = make_double2(uz, w);
                Bin.idp[o] = make_ulonglong2(cpid, (pk & 0x00000000FFFFFFFFull) | ((uint64_t)(uint32_t)cg << 32));
              }
            }
            if (defer) n_new = 0;                            // (their first child still takes the parent's slot)
          }
        }
        // families that fit: unborn children (parent id, flight counter and child index) into free slots
        uint32_t ifit = n_new;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const uint32_t t = __shfl_up_sync(0xffffffffu, ifit, o);
          if (lane >= o) ifit += t;
        }
        const uint32_t take = __shfl_sync(0xffffffffu, ifit, 31);
        if (n_new) {
          const double2 a2 = s_xy[slot], b2 = s_zt[slot];
          const int mm = s_mat[slot] & 0xFFFF;
          for (uint32_t j = 1; j <= n_new; ++j) {
            const uint32_t cs = l_free[nFree - 1u - (ifit - n_new + j - 1u)];
            s_xy[cs] = a2; s_zt[cs] = b2; s_uzw[cs] = make_double2(0.0, w);
            s_idp[cs] = make_ulonglong2(pid, pk);
            s_mat[cs] = mm | (int)(j << 16);
          }
        }
        __syncwarp();
        for (uint32_t k = lane; k < take; k += 32) l_b[nB + k] = l_free[nFree - 1u - k];
        nB += take; nFree -= take;
      }
      const bool scat = active && kind == 1, born = active && kind == 2 && n_out > 0u;
      const unsigned b1 = __ballot_sync(0xffffffffu, scat);
      const unsigned b2 = __ballot_sync(0xffffffffu, born);
      if (scat) l_f[nF + __popc(b1 & lt_mask)] = (uint8_t)slot;
      if (born) l_b[nB + __popc(b2 & lt_mask)] = (uint8_t)slot;      // child 0 in the parent's slot
      nF += __popc(b1); nB += __popc(b2);
      if (active && kind != 3) {
        ++c_coll;
        if (kind == 1) ++c_scat; else if (kind == 0) ++c_capt; else { ++c_fis; c_sec += n_out; }
      }
      __syncwarp();
      ring_push(active && (kind == 0 || kind == 2), pid, ectr, kind == 0 ? END_CAPTURE : END_FISSION);
    } else {
      // ================= birth round (A10): id, group and direction of fission children =================
      blocked = false;
      const uint32_t cnt = min(nB, 32u);
      const bool active = (uint32_t)lane < cnt;
      if (active) {
        const uint32_t slot = l_b[nB - 1u - lane];
        const ulonglong2 id = s_idp[slot];                   // still the parent's id and packed state
        const int mm = s_mat[slot];
        const double w = s_uzw[slot].y;
        const int m = mm & 0xFF;
        const U4 rc = draw_block(id.x, pk_ectr(id.y), BLK_CHILD + (uint32_t)(mm >> 16), seedb);
        const uint64_t cpid = (1ull << 63) | ((((uint64_t)rc.x << 32) | (uint64_t)rc.y) >> 1);
        const U4 rg = draw_block(cpid, 0, BLK_SRC_ZG, seedb);
        const int cg = sample_cdf(T.cdf_chi + m * G, G, u52(rg.z, rg.w));
        const U4 rd = draw_block(cpid, 0, BLK_SRC_DIR, seedb);
        double ux, uy, uz;
        isotropic_dir(u52(rd.x, rd.y), u52(rd.z, rd.w), ux, uy, uz);
        s_uxy[slot] = make_double2(ux, uy);
        s_uzw[slot] = make_double2(uz, w);
        s_idp[slot] = make_ulonglong2(cpid, (id.y & 0x00000000FFFFFFFFull) | ((uint64_t)(uint32_t)cg << 32));
        s_mat[slot] = mm & 0xFFFF;
        l_f[nF + lane] = (uint8_t)slot;
      }
      nB -= cnt; nF += cnt;
      __syncwarp();
    }
  }
  if ((uint32_t)lane < nH) fp += end_hash(h_pid[lane], h_ce[lane] & 0xFFFFFFu, (int)(h_ce[lane] >> 24));

  warp_count(s_cnt, K_FLIGHTS, c_flights);
  warp_count(s_cnt, K_SEGMENTS, c_segments);
  warp_count(s_cnt, K_CROSSINGS, c_cross);
  warp_count(s_cnt, K_REFLECTIONS, c_refl);
  warp_count(s_cnt, K_LEAKS, c_leak);
  warp_count(s_cnt, K_CENSUS, c_census);
  warp_count(s_cnt, K_LOST, c_lost);
  warp_count(s_cnt, K_COLLISIONS, c_coll);
  warp_count(s_cnt, K_SCATTERS, c_scat);
  warp_count(s_cnt, K_CAPTURES, c_capt);
  warp_count(s_cnt, K_FISSIONS, c_fis);
  warp_count(s_cnt, K_SECONDARIES, c_sec);
  warp_count64(s_cnt, K_FINGERPRINT, fp);
  flush_counts(s_cnt, ctl->cnt);
}

// after a pool launch: fission children that found the pools full sit behind the processed range
// (the spill window [spill_lo, bank_tail)); they become the next range, and the next spill window is
// the free part of the bank on the other side of it
__global__ void k_pool_begin(Ctl *ctl, uint32_t capacity)
{
  ctl->fetch = 0u; ctl->bank_tail = ctl->n_active; ctl->spill_lo = ctl->n_active; ctl->spill_limit = capacity;
}
__global__ void k_pool_next(Ctl *ctl, uint32_t *mirror, uint32_t capacity)
{
  const uint32_t lo = ctl->spill_lo, hi = ctl->overflow ? lo : ctl->bank_tail;
  ctl->fetch = lo;
  ctl->n_active = hi;
  if (lo == 0u) { ctl->spill_lo = hi; ctl->bank_tail = hi; ctl->spill_limit = capacity; }
  else { ctl->spill_lo = 0u; ctl->bank_tail = 0u; ctl->spill_limit = lo; }
  ctl->iter += 1u;
  mirror[0] = hi - lo; mirror[1] = ctl->n_census; mirror[2] = ctl->overflow; mirror[3] = hi;
  mirror[4] = (uint32_t)ctl->cnt[K_FLIGHTS]; mirror[5] = (uint32_t)(ctl->cnt[K_FLIGHTS] >> 32);
}

}  // namespace mcdc
