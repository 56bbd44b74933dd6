// mcdc_comb.cu — census close: canonical ordering of the
// census bank by particle id, the uniform-weight population comb, and the batch
// close-out of the tally.  Definitions: DESIGN.md §3 C.8, C.9.
//
// Ordering.  Particle ids fall in three classes ordered by their top bits: source
// ids (dense 0..N-1), comb-survivor ids (dense j under a fixed step tag) and fission
// children (uniformly hashed 63-bit ids).  A monotone bucket function maps ids to
// ~n/4 buckets; a counting sort (histogram, scan, scatter) groups the census list by
// bucket and one thread per bucket finishes the order on the full key
// (pid, then the bit patterns of t, x, y, z).  Monotone buckets + sorted buckets =
// globally sorted list, independent of the slot order the event kernels produced.
#include "mcdc_kernels.cuh"

namespace mcdc {

struct BucketMap {
  uint32_t shift_dense;      // dense ids: bucket = id >> shift_dense
  uint32_t nb0, nb1;         // buckets of class 00 (source) and 01 (comb survivors)
  uint32_t bits_hash;        // children: bucket = top bits_hash bits of the 63-bit hash
  unsigned long long base1;  // (k << 40) of the survivors alive in this step
  uint32_t n_buckets;
};

static __device__ __forceinline__ uint32_t bucket_of(const BucketMap &M, unsigned long long pid)
{
  const unsigned cls = (unsigned)(pid >> 62);
  if (cls == 0u) {
    const unsigned long long b = pid >> M.shift_dense;
    return (uint32_t)(b < M.nb0 ? b : M.nb0 - 1);
  }
  if (cls == 1u) {
    const unsigned long long low = pid & 0x3FFFFFFFFFFFFFFFull;
    const unsigned long long rel = low > M.base1 ? low - M.base1 : 0ull;
    const unsigned long long b = rel >> M.shift_dense;
    return M.nb0 + (uint32_t)(b < M.nb1 ? b : M.nb1 - 1);
  }
  return M.nb0 + M.nb1 + (uint32_t)((pid & 0x7FFFFFFFFFFFFFFFull) >> (63u - M.bits_hash));
}

// (reads the id array only; the uniform-weight check of C.8 step 2 is made by k_comb on the records it takes)
__global__ void __launch_bounds__(BS) k_bucket_hist(BucketMap M, Bank B, const uint32_t *__restrict__ list,
                                                    const Ctl *ctl, uint32_t *__restrict__ count)
{
  const uint32_t n = ctl->n_census;
  if (n == 0u || ctl->overflow) return;      // (overflow: the census list is incomplete, n may exceed the capacity)
  for (uint32_t i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS)
    atomicAdd(count + bucket_of(M, B.idp[list[i]].x), 1u);
}

// exclusive scan of count[0..n) in three phases (block sums, scan of sums, apply)
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = BS * SCAN_ITEMS;

static __device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *s_w, uint32_t &total)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_w[wid] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
    for (int w = 0; w < NWARP; ++w) { const uint32_t c = s_w[w]; s_w[w] = run; run += c; }
    s_w[NWARP] = run;
  }
  __syncthreads();
  const uint32_t r = s_w[wid] + incl - v;
  total = s_w[NWARP];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(BS) k_scan_tiles(const uint32_t *__restrict__ in, uint32_t n,
                                                   uint32_t *__restrict__ tile_sum)
{
  __shared__ uint32_t s_w[NWARP + 1];
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) s += in[base + k];
  uint32_t total;
  block_exclusive_scan(s, s_w, total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(BS) k_scan_sums(uint32_t *tile_sum, uint32_t n_tiles)
{
  __shared__ uint32_t s_w[NWARP + 1];
  uint32_t carry = 0;
  for (uint32_t base = 0; base < n_tiles; base += BS) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < n_tiles ? tile_sum[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, s_w, total);
    if (i < n_tiles) tile_sum[i] = carry + ex;
    carry += total;
  }
}

__global__ void __launch_bounds__(BS) k_scan_apply(const uint32_t *__restrict__ in, uint32_t n,
                                                   const uint32_t *__restrict__ tile_sum,
                                                   uint32_t *__restrict__ offs, uint32_t *__restrict__ cursor)
{
  __shared__ uint32_t s_w[NWARP + 1];
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? in[base + k] : 0u; s += v[k]; }
  uint32_t total;
  uint32_t run = tile_sum[blockIdx.x] + block_exclusive_scan(s, s_w, total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < n) { offs[base + k] = run; cursor[base + k] = run; run += v[k]; }
}

__global__ void __launch_bounds__(BS) k_bucket_scatter(BucketMap M, Bank B, const uint32_t *__restrict__ list,
                                                       const Ctl *ctl, uint32_t *__restrict__ cursor,
                                                       uint32_t *__restrict__ order)
{
  const uint32_t n = ctl->overflow ? 0u : ctl->n_census;
  for (uint32_t i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS) {
    const uint32_t slot = list[i];
    order[atomicAdd(cursor + bucket_of(M, B.idp[slot].x), 1u)] = slot;
  }
}

// order of two census entries: id first; equal ids (hashed child ids can collide) by the bit
// patterns of t, x, y, z, which are only loaded in that case
static __device__ __forceinline__ bool entry_less(const Bank &B, unsigned long long pa, uint32_t sa,
                                                  unsigned long long pb, uint32_t sb)
{
  if (pa != pb) return pa < pb;
  const double2 xa = B.xy[sa], za = B.zt[sa], xb = B.xy[sb], zb = B.zt[sb];
  const unsigned long long ka[4] = {(unsigned long long)__double_as_longlong(za.y), (unsigned long long)__double_as_longlong(xa.x),
                                    (unsigned long long)__double_as_longlong(xa.y), (unsigned long long)__double_as_longlong(za.x)};
  const unsigned long long kb[4] = {(unsigned long long)__double_as_longlong(zb.y), (unsigned long long)__double_as_longlong(xb.x),
                                    (unsigned long long)__double_as_longlong(xb.y), (unsigned long long)__double_as_longlong(zb.x)};
#pragma unroll
  for (int i = 0; i < 4; ++i) if (ka[i] != kb[i]) return ka[i] < kb[i];
  return false;
}

// one thread per bucket: insertion sort of its (short) run on the full key
__global__ void __launch_bounds__(BS) k_bucket_sort(Bank B, const uint32_t *__restrict__ offs,
                                                    const uint32_t *__restrict__ cursor, uint32_t n_buckets,
                                                    uint32_t *__restrict__ order)
{
  for (uint32_t b = blockIdx.x * BS + threadIdx.x; b < n_buckets; b += gridDim.x * BS) {
    const uint32_t lo = offs[b], hi = cursor[b];     // cursor = end of the bucket after the scatter
    for (uint32_t i = lo + 1; i < hi; ++i) {
      const uint32_t si = order[i];
      const unsigned long long pi = B.idp[si].x;
      uint32_t j = i;
      while (j > lo) {
        const uint32_t sj = order[j - 1];
        if (!entry_less(B, pi, si, B.idp[sj].x, sj)) break;
        order[j] = sj; --j;
      }
      order[j] = si;
    }
  }
}

// A12 comb: tooth j takes sorted entry floor((j + a) N / M), weight w N / M, new id.
// Where a survivor is written does not matter to any result (ids come from the tooth index), so the
// bank is filled from both ends: survivors whose group has many mean free paths ahead of it in the
// next census step (vsig[g] = v_g * max sigma_t_g >= min_vsig) from the front, the rest from the
// back.  The pool kernel deals the bank in order, so long histories start first and do not end the
// launch alone.  One atomic per block and end (ballot/popc ranks inside the block).
__global__ void __launch_bounds__(BS) k_comb(Bank src, Bank dst, const uint32_t *__restrict__ order,
                                             Ctl *ctl, uint32_t *__restrict__ q_active,
                                             unsigned long long M, const double *__restrict__ vsig,
                                             double min_vsig, int unit_w /* C.14: a generation starts with weight 1 */,
                                             uint32_t *flag /* [0]: the census weights are not uniform (C.8 step 2) */)
{
  __shared__ uint32_t s_w[NWARP + 1];
  const unsigned long long N = ctl->n_census;
  if (N == 0ull || ctl->overflow) return;
  // comb offset of this census step: its own Philox stream (C.1)
  const unsigned long long seedb = ctl->seedb;
  const U4 ro = philox4x32_10(0xFFFFFFFFu, 0xFFFFFFFFu, ctl->step_k1, 0u, (uint32_t)seedb,
                              (uint32_t)(seedb >> 32));
  const double a = u52(ro.x, ro.y);
  const unsigned long long id_tag = (1ull << 62) | ((unsigned long long)ctl->step_k1 << 40);
  const double r = (double)N / (double)M;
  const double w0 = src.uzw[order[0]].y;               // every record the comb takes must carry this weight
  for (unsigned long long base = blockIdx.x * (unsigned long long)BS; base < M;
       base += (unsigned long long)gridDim.x * BS) {
    const unsigned long long j = base + threadIdx.x;
    const bool valid = j < M;
    uint32_t s = 0;
    ulonglong2 id = make_ulonglong2(0ull, 0ull);
    bool lng = false;
    if (valid) {
      const double pos = ((double)j + a) * r;
      unsigned long long idx = (unsigned long long)pos;
      if (idx > N - 1ull) idx = N - 1ull;
      s = order[idx];
      id = src.idp[s];
      lng = __ldg(vsig + pk_g(id.y)) >= min_vsig;
    }
    const uint32_t pf = block_reserve1(valid && lng, &ctl->comb_front, s_w);
    const uint32_t pb = block_reserve1(valid && !lng, &ctl->comb_back, s_w);
    if (valid) {
      const uint32_t o = lng ? pf : (uint32_t)(M - 1ull) - pb;
      const double2 e2 = src.uzw[s];
      if (e2.y != w0) *flag = 1u;
      dst.xy[o] = src.xy[s];
      dst.zt[o] = src.zt[s];
      dst.uxy[o] = src.uxy[s];
      dst.uzw[o] = make_double2(e2.x, unit_w ? 1.0 : e2.y * r);
      dst.idp[o] = make_ulonglong2(id_tag | j, id.y & 0x000000FFFFFFFFFFull);   // ectr = 0
      q_active[o] = o;
    }
  }
}

// ---- weighted comb (C.15; "population control techniques [9,10]") ----
// Weights become fixed-point integers q = floor(w 2^32 + 1/2); their prefix sums over the canonical
// order are exact integers, so the teeth are the same whatever the order of summation (the parallel
// scan below and a sequential loop agree bit for bit).  Tooth j sits at floor((j + a) W_q / M) on the
// axis of cumulated weights and takes the entry whose interval holds it; every survivor weighs W / M.
__global__ void __launch_bounds__(BS) k_wq(Bank B, const uint32_t *__restrict__ order, const Ctl *ctl,
                                           unsigned long long *__restrict__ q, uint32_t *flag)
{
  const uint32_t n = ctl->overflow ? 0u : ctl->n_census;
  for (uint32_t i = blockIdx.x * BS + threadIdx.x; i < n; i += gridDim.x * BS) {
    const double w = B.uzw[order[i]].y;
    const bool ok = w >= 0.0 && w < 524288.0;
    if (!ok) flag[1] = 1u;
    q[i] = ok ? (unsigned long long)(w * 4294967296.0 + 0.5) : 0ull;
  }
}

static __device__ __forceinline__ unsigned long long block_exclusive_scan64(unsigned long long v, unsigned long long *s_w,
                                                                            unsigned long long &total)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  unsigned long long incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_w[wid] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long run = 0;
    for (int w = 0; w < NWARP; ++w) { const unsigned long long c = s_w[w]; s_w[w] = run; run += c; }
    s_w[NWARP] = run;
  }
  __syncthreads();
  const unsigned long long r = s_w[wid] + incl - v;
  total = s_w[NWARP];
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(BS) k_scan64_tiles(const unsigned long long *__restrict__ in, const Ctl *ctl,
                                                     unsigned long long *__restrict__ tile_sum)
{
  __shared__ unsigned long long s_w[NWARP + 1];
  const uint32_t n = ctl->overflow ? 0u : ctl->n_census;
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  unsigned long long s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) if (base + k < n) s += in[base + k];
  unsigned long long total;
  block_exclusive_scan64(s, s_w, total);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = total;
}

// exclusive scan of the tile sums; the grand total goes behind the n prefixes (pre[n]) and flags an
// overflow of the fixed-point sum
__global__ void __launch_bounds__(BS) k_scan64_sums(unsigned long long *tile_sum, uint32_t n_tiles, const Ctl *ctl,
                                                    unsigned long long *pre, uint32_t *flag)
{
  __shared__ unsigned long long s_w[NWARP + 1];
  unsigned long long carry = 0;
  for (uint32_t base = 0; base < n_tiles; base += BS) {
    const uint32_t i = base + threadIdx.x;
    const unsigned long long v = i < n_tiles ? tile_sum[i] : 0ull;
    if (v >> 62) flag[1] = 1u;
    unsigned long long total;
    const unsigned long long ex = block_exclusive_scan64(v, s_w, total);
    if (i < n_tiles) tile_sum[i] = carry + ex;
    carry += total;
    if (carry >> 62) flag[1] = 1u;
  }
  if (threadIdx.x == 0 && !ctl->overflow) pre[ctl->n_census] = carry;
}

__global__ void __launch_bounds__(BS) k_scan64_apply(unsigned long long *__restrict__ q, const Ctl *ctl,
                                                     const unsigned long long *__restrict__ tile_sum)
{
  __shared__ unsigned long long s_w[NWARP + 1];
  const uint32_t n = ctl->overflow ? 0u : ctl->n_census;
  const uint32_t base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  unsigned long long v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { v[k] = (base + k < n) ? q[base + k] : 0ull; s += v[k]; }
  unsigned long long total;
  unsigned long long run = tile_sum[blockIdx.x] + block_exclusive_scan64(s, s_w, total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < n) { q[base + k] = run; run += v[k]; }      // in place: a tile reads its items before it writes
}

__global__ void __launch_bounds__(BS) k_comb_weighted(Bank src, Bank dst, const uint32_t *__restrict__ order,
                                                      const unsigned long long *__restrict__ pre, Ctl *ctl,
                                                      uint32_t *__restrict__ q_active, unsigned long long M)
{
  const unsigned long long N = ctl->n_census;
  if (N == 0ull || ctl->overflow) return;
  const unsigned long long Wq = pre[N];
  if (Wq == 0ull) return;                              // nothing but zero weights: no survivors (k_end_step)
  const unsigned long long seedb = ctl->seedb;
  const U4 ro = philox4x32_10(0xFFFFFFFFu, 0xFFFFFFFFu, ctl->step_k1, 0u, (uint32_t)seedb, (uint32_t)(seedb >> 32));
  const double a = u52(ro.x, ro.y);
  const unsigned long long id_tag = (1ull << 62) | ((unsigned long long)ctl->step_k1 << 40);
  const double r = (double)Wq / (double)M;
  const double w_out = ((double)Wq * (1.0 / 4294967296.0)) / (double)M;
  for (unsigned long long j = blockIdx.x * (unsigned long long)BS + threadIdx.x; j < M;
       j += (unsigned long long)gridDim.x * BS) {
    const double pos = ((double)j + a) * r;
    unsigned long long t = (unsigned long long)pos;
    if (t > Wq - 1ull) t = Wq - 1ull;
    unsigned long long lo = 0, hi = N;                 // pre[lo] <= t < pre[hi]
    while (hi - lo > 1ull) { const unsigned long long mid = lo + (hi - lo) / 2ull; if (pre[mid] <= t) lo = mid; else hi = mid; }
    const uint32_t s = order[lo];
    const ulonglong2 id = src.idp[s];
    const double2 e2 = src.uzw[s];
    const uint32_t o = (uint32_t)j;
    dst.xy[o] = src.xy[s];
    dst.zt[o] = src.zt[s];
    dst.uxy[o] = src.uxy[s];
    dst.uzw[o] = make_double2(e2.x, w_out);
    dst.idp[o] = make_ulonglong2(id_tag | j, id.y & 0x000000FFFFFFFFFFull);   // ectr = 0
    q_active[o] = o;
  }
}

// census without combing: gather the census bank into fresh contiguous slots so that
// dead slots are reclaimed at every census (ids, weights and flight counters kept)
__global__ void __launch_bounds__(BS) k_census_gather(Bank src, Bank dst, const uint32_t *__restrict__ list,
                                                      const Ctl *ctl, uint32_t *__restrict__ q_active)
{
  const uint32_t n = ctl->overflow ? 0u : ctl->n_census;
  for (uint32_t j = blockIdx.x * BS + threadIdx.x; j < n; j += gridDim.x * BS) {
    const uint32_t s = list[j];
    dst.xy[j] = src.xy[s]; dst.zt[j] = src.zt[s]; dst.uxy[j] = src.uxy[s];
    dst.uzw[j] = src.uzw[s]; dst.idp[j] = src.idp[s];
    q_active[j] = j;
  }
}

// mid-step bank compaction (keeps fission chains from exhausting the bank): live
// particles = active queue + census list; both are gathered into the other bank and
// the lists rewritten in place as contiguous ranges
__global__ void __launch_bounds__(BS) k_compact(Bank src, Bank dst, uint32_t *__restrict__ q_active,
                                                uint32_t *__restrict__ q_census, const Ctl *ctl)
{
  const uint32_t na = ctl->n_active, nc = ctl->n_census;
  for (uint32_t j = blockIdx.x * BS + threadIdx.x; j < na + nc; j += gridDim.x * BS) {
    uint32_t *e = j < na ? q_active + j : q_census + (j - na);
    const uint32_t s = *e;
    dst.xy[j] = src.xy[s]; dst.zt[j] = src.zt[s]; dst.uxy[j] = src.uxy[s];
    dst.uzw[j] = src.uzw[s]; dst.idp[j] = src.idp[s];
    *e = j;
  }
}
__global__ void k_compact_done(Ctl *ctl, uint32_t *mirror)
{
  ctl->bank_tail = ctl->n_active + ctl->n_census;
  mirror[3] = ctl->bank_tail;
}

// A14 batch close-out: fold the batch tally into the running sums
// (the first close-out of a run writes the sums instead of adding to them: no separate zeroing pass)
__global__ void __launch_bounds__(BS) k_closeout(const double *__restrict__ batch, double *__restrict__ sum1,
                                                 double *__restrict__ sum2, size_t n, int first)
{
  for (size_t i = blockIdx.x * (size_t)BS + threadIdx.x; i < n; i += (size_t)gridDim.x * BS) {
    const double b = batch[i];
    if (first) { sum1[i] = b; sum2[i] = b * b; }
    else { sum1[i] += b; sum2[i] += b * b; }
  }
}

// mean / standard error over batches (mcdc_tally_read which = 0, 1)
__global__ void __launch_bounds__(BS) k_tally_stats(const double *__restrict__ sum1, const double *__restrict__ sum2,
                                                    double *__restrict__ out, size_t n, double n_batch,
                                                    double n_hist, int which)
{
  for (size_t i = blockIdx.x * (size_t)BS + threadIdx.x; i < n; i += (size_t)gridDim.x * BS) {
    if (which == 0) out[i] = sum1[i] / (n_batch * n_hist);
    else if (n_batch < 2.0) out[i] = 0.0;
    else {
      const double mean = sum1[i] / n_batch;
      double var = (sum2[i] / n_batch - mean * mean) * (n_batch / (n_batch - 1.0));
      if (var < 0.0) var = 0.0;
      out[i] = sqrt(var / n_batch) / n_hist;
    }
  }
}

}  // namespace mcdc
