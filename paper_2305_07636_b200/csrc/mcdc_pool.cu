// mcdc_pool.cu — one census step of the history loop as ONE persistent launch
// (SURVEY §8(a) rows A0, A2-A11, A13).  Definitions: DESIGN.md §3; design: DESIGN.md §6.
//
// Every warp keeps a pool of PW particles in shared memory (80-byte records + material) and
// lists of pool slots by next event: flight-ready, collision-ready (which includes fission
// children waiting to be born), waiting for the census write-out, free.  A round takes up to
// 32 slots of ONE list, so all lanes of the warp run the same event code (the divergence
// between flying and colliding particles that the paper hands to an asynchronous scheduler,
// PAPER.md:51, is removed by construction).  Particles enter the pool from the dense active
// bank (coalesced 128-bit loads, ranges reserved with one atomic per warp and chunk) and leave
// it either dead or through the census write-out (32 records at a time, one atomic, coalesced
// 128-bit stores into the other bank).  Between entry and exit a particle never touches HBM;
// only tally adds and the material map do.
// Fission children take free pool slots as unborn records (parent id, flight counter, child
// index); their id, group and direction are drawn in a later collision-kind round, by the
// same three Philox sites a scatter uses.  A fission whose children do not fit is retried
// later (the counter-based RNG makes the retry identical); only when a pool holds nothing but
// such parents are unborn children appended to the active bank behind the range being
// processed, and the host relaunches over that range.  Terminal events are hashed into the
// fingerprint 32 at a time from a ring, as a round kind of its own.
#include "mcdc_kernels.cuh"

namespace mcdc {

#ifndef POOL_PW
#define POOL_PW 112                // pool slots per warp (<= 256: lists are bytes)
#endif
#ifndef POOL_RESERVE
#define POOL_RESERVE 16            // pool slots kept free for fission children when particles are dealt in
#endif
#ifndef MB_POOL
#define MB_POOL 2
#endif
#ifndef POOL_PHASE_SHIFT
#define POOL_PHASE_SHIFT 14        // plain general variants: period (log2 SM clocks) of the flight / collision phases
#endif
#ifndef POOL_PHASE_MIN
#define POOL_PHASE_MIN 24          // ... and the list length from which a warp follows the phase
#endif
#ifndef POOL_NT
#define POOL_NT 256                // threads per block
#endif
constexpr int PW = POOL_PW;
constexpr int POOL_THREADS = POOL_NT;
constexpr int POOL_WARPS = POOL_THREADS / 32;
constexpr int HRING = 64;                              // terminal events waiting for their fingerprint hash
constexpr int POOL_BYTES = PW * (80 + 4) + 4 * PW + HRING * 12;   // records, material, four byte lists, hash ring
static_assert(POOL_BYTES % 16 == 0, "pool alignment");
// MARCH variants (tally mesh finer than the lattice): 24 bytes per slot to suspend a tally march (flight length, last
// crossing distance, four 16-bit tally indices) and the list of suspended flights
constexpr int POOL_MARCH_BYTES = PW * 24 + PW;
static_assert(POOL_MARCH_BYTES % 16 == 0, "pool alignment");
static __host__ __device__ __forceinline__ constexpr int pool_bytes(bool march) { return POOL_BYTES + (march ? POOL_MARCH_BYTES : 0); }
#ifndef MARCH_MIN
#define MARCH_MIN 12               // marching lanes below which the rest of a march is suspended and regrouped
#endif
#ifndef MARCH_ITER_MIN
#define MARCH_ITER_MIN 4           // iterations a round of resumed marches runs at least
#endif
#ifndef MARCH_FIRST
#define MARCH_FIRST 2              // iterations a round of fresh flights runs at least
#endif
// segments per flight (counted on the finished batches) from which the MARCH variants are taken: below, the
// marches are too short to pay for a suspension.  Measured: config 4 (1.5 segments per flight)
// -8 %, eigenvalue pin cell (4.3) -15 %, dog-leg duct (6.6) +4 %, config 2 (12) +33 %.
constexpr double MARCH_SEGMENTS_PER_FLIGHT = 6.0;
static_assert(PW >= 64 && PW <= 256 && POOL_RESERVE + 32 <= PW, "pool size");

// bits of the per-slot material word: material | (pin material + 1) << 8 | child index << 16 | unborn << 24
// | event << 25 | surface << 27 of a suspended flight (MARCH)
constexpr int MAT_UNBORN = 1 << 24;
constexpr int MAT_UNKNOWN = 0xFF;   // lean variants: material of a particle that has just entered a lattice cell (n_mat <= 127)

static __host__ __device__ __forceinline__ size_t pool_table_bytes(const TableLayout &L, int use_smem)
{
  return use_smem ? (((size_t)L.total * 8 + 15) & ~(size_t)15) : 0;
}
static __host__ __device__ __forceinline__ size_t pool_plane_bytes(int nx, int ny, int nz, int n_mat, int G)
{
  // plane tables + first non-zero entry of every scatter CDF row (bytes) + for G <= 8 the rows as eight fp32 thresholds
  return ((((size_t)(nx + ny + nz + 3) * 8) + (size_t)n_mat * G + 15) & ~(size_t)15) + (G <= 8 ? (size_t)n_mat * G * 32 : 0);
}
// MARCH variants keep the tally plane tables in shared memory too: a step of the march waits for one plane
static __host__ __device__ __forceinline__ size_t pool_csg_bytes(int n_surf) { return (size_t)n_surf * 80; }
static __host__ __device__ __forceinline__ size_t pool_tally_plane_bytes(int tnx, int tny, int tnz, int tnt, bool march)
{
  return march ? (((size_t)(tnx + tny + tnz + tnt + 4) * 8 + 15) & ~(size_t)15) : 0;
}

static __device__ __forceinline__ int mat_pack(int m, int pin) { return (m & 0xFF) | ((pin + 1) << 8); }

// distance to the plane the particle is heading to, from the two planes of its interval (C.5, App. C)
static __device__ __forceinline__ double plane_dist2(double lo, double hi, double p, double u)
{
  if (u == 0.0) return __longlong_as_double(0x7FF0000000000000ll);
  const double d = ((u > 0.0 ? hi : lo) - p) / u;
  return d < 0.0 ? 0.0 : d;
}

// The tally march of ONE flight by one lane on its own (App. C.2; same steps, same arithmetic and same order of the
// adds per flight as the warp-synchronous march in k_pool): the fallback of the POOL_LEAN variants.  Not inlined: its
// registers and code stay out of the hot loop.  Returns the scored segments, bit 31 set when the flight left the tally
// mesh (lost); fxyz = the spatial tally bin the flight ends in.
struct MarchTables {               // what march_alone needs of the problem (built at the call, which is rare)
  const double *tx, *ty, *tz, *tt;
  int tnx, tny, tnz, tnt;
  AxisHint hx, hy, hz, ht;
  double *tally;
  long long tcross_off;
};
template <bool TC>
static __device__ __noinline__ uint32_t march_alone(const MarchTables P, int G, double x, double y, double z, double t,
                                                    double ux, double uy, double uz, double w, double v, double d,
                                                    int g, int *fxyz)
{
  const double INF = __longlong_as_double(0x7FF0000000000000ll);
  int jx = find_interval_fast(P.tx, P.tnx, x, ux, P.hx);
  int jy = find_interval_fast(P.ty, P.tny, y, uy, P.hy);
  int jz = find_interval_fast(P.tz, P.tnz, z, uz, P.hz);
  int jt = find_interval_fast(P.tt, P.tnt, t, 1.0, P.ht);
  double sx = plane_dist(P.tx, jx, x, ux), sy = plane_dist(P.ty, jy, y, uy), sz = plane_dist(P.tz, jz, z, uz);
  double st = (__ldg(P.tt + jt + 1) - t) * v; if (st < 0.0) st = 0.0;
  const long long st_y = P.tnx, st_z = (long long)P.tny * P.tnx, st_t = (long long)G * P.tnz * P.tny * P.tnx;
  long long cur = ((((long long)jt * G + g) * P.tnz + jz) * P.tny + jy) * P.tnx + jx;
  double s_prev = 0.0;
  uint32_t nseg = 0;
  bool lost = false;
  for (;;) {
    int axis = 0; double s_min = sx;
    if (sy < s_min) { s_min = sy; axis = 1; }
    if (sz < s_min) { s_min = sz; axis = 2; }
    if (st < s_min) { s_min = st; axis = 3; }
    const bool cross = s_min < d;
    const double len = (cross ? s_min : d) - s_prev;
    if (len > 0.0) { atomicAdd(P.tally + cur, w * len); ++nseg; }
    if (!cross) break;
    const bool spatial = axis < 3;
    const double ua = axis == 0 ? ux : axis == 1 ? uy : uz;
    const double pa = axis == 0 ? x : axis == 1 ? y : z;
    const double *const Pa = axis == 0 ? P.tx : axis == 1 ? P.ty : axis == 2 ? P.tz : P.tt;
    const int na = axis == 0 ? P.tnx : axis == 1 ? P.tny : axis == 2 ? P.tnz : P.tnt;
    const int jo = axis == 0 ? jx : axis == 1 ? jy : axis == 2 ? jz : jt;
    const bool up = !spatial || ua > 0.0;
    const int ja = jo + (up ? 1 : -1);
    const bool out = ja < 0 || ja >= na;
    const double edge = __ldg(Pa + (out ? 0 : ja + (up ? 1 : 0)));
    double sa = spatial ? (edge - pa) / ua : (edge - t) * v;
    if (sa < 0.0) sa = 0.0;
    if (out) { lost = true; sa = INF; }
    if (TC && !spatial) atomicAdd(P.tally + P.tcross_off + cur, w * v);     // C.13: the time passes a tally time edge
    cur += axis == 0 ? (long long)(up ? 1 : -1) : axis == 1 ? (up ? st_y : -st_y) : axis == 2 ? (up ? st_z : -st_z) : st_t;
    jx = axis == 0 ? ja : jx; jy = axis == 1 ? ja : jy; jz = axis == 2 ? ja : jz; jt = axis == 3 ? ja : jt;
    sx = axis == 0 ? sa : sx; sy = axis == 1 ? sa : sy; sz = axis == 2 ? sa : sz; st = axis == 3 ? sa : st;
    s_prev = s_min;
    if (lost) break;
  }
  fxyz[0] = jx; fxyz[1] = jy; fxyz[2] = jz;
  return nseg | (lost ? 0x80000000u : 0u);
}

// Distance to the nearest of the three planes the particle is heading to and its axis (C.5): the smallest of
// ((u > 0 ? hi : lo) - p) / u over x, y, z, the earlier axis on a tie.  Only the smallest quotient is needed, so the
// axes are first RANKED without dividing — e_x / u_x < e_y / u_y iff |e_x| |u_y| < |e_y| |u_x| — and one division
// gives the winner's distance, the very operation of the definition.  The ranking is trusted only where it is certain
// for the ROUNDED quotients: the products must differ by more than 2^-48 relative (each carries one rounding of 2^-53;
// quotients whose exact values differ by 2^-49 relative round to different, equally ordered doubles); numerators and
// directions must agree in sign (else the definition clamps a negative distance to 0) and everything must be finite.
// Any other case — a particle on two planes at once, a direction cosine of exactly 0 beside another, an infinite
// plane — takes the three divisions of the definition.
static __device__ __forceinline__ double nearest_plane(double lx, double hx, double ly, double hy, double lz, double hz,
                                                       double x, double y, double z, double ux, double uy, double uz,
                                                       bool finite, int &surf)
{
  const double ex = (ux > 0.0 ? hx : lx) - x, ey = (uy > 0.0 ? hy : ly) - y, ez = (uz > 0.0 ? hz : lz) - z;
  if (finite) {
    constexpr double EPS = 3.552713678800501e-15 /* 2^-48 */, TINY = 1e-290;
    const int sgn = (__double2hiint(ex) ^ __double2hiint(ux)) | (__double2hiint(ey) ^ __double2hiint(uy)) |
                    (__double2hiint(ez) ^ __double2hiint(uz));
    const double pxy = fabs(ex) * fabs(uy), pyx = fabs(ey) * fabs(ux);
    const double d1 = pxy - pyx;                              // > 0: y is nearer than x
    bool sure = fabs(d1) > fma(EPS, pxy + pyx, TINY);
    const bool yn = d1 > 0.0;
    double ew = yn ? ey : ex, uw = yn ? uy : ux;
    const double pwz = fabs(ew) * fabs(uz), pzw = fabs(ez) * fabs(uw);
    const double d2 = pwz - pzw;                              // > 0: z is nearer than the winner of x, y
    sure = sure && fabs(d2) > fma(EPS, pwz + pzw, TINY);
    const bool zn = d2 > 0.0;
    ew = zn ? ez : ew; uw = zn ? uz : uw;
    if (sure && sgn >= 0) { surf = zn ? 2 : yn ? 1 : 0; return ew / uw; }
  }
  const double dsx = plane_dist2(lx, hx, x, ux), dsy = plane_dist2(ly, hy, y, uy), dsz = plane_dist2(lz, hz, z, uz);
  double d_s = dsx; surf = 0;
  if (dsy < d_s) { d_s = dsy; surf = 1; }
  if (dsz < d_s) { d_s = dsz; surf = 2; }
  return d_s;
}

// One Philox block behind a call: the general variants (whose hot code does not fit the 32 KB instruction cache of an
// SM, profiles/pool_dogleg_r2.md) share one copy among their call sites; the lean variants inline theirs.
static __device__ __noinline__ U4 philox_shared(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3)
{
  return philox4x32_10(k0, k1, c0, c1, c2, c3);
}
// (likewise the clamped plane distance e / u of C.5 and a plain division)
static __device__ __noinline__ double ratio_shared(double e, double u)
{
  if (u == 0.0) return __longlong_as_double(0x7FF0000000000000ll);
  const double d = e / u;
  return d < 0.0 ? 0.0 : d;
}
static __device__ __noinline__ double div_shared(double a, double b) { return a / b; }
template <bool SHARED>
static __device__ __forceinline__ U4 philox_site(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3)
{
  return SHARED ? philox_shared(k0, k1, c0, c1, c2, c3) : philox4x32_10(k0, k1, c0, c1, c2, c3);
}

// TC: the tally carries the time-crossing block (C.13); compiled out of the default kernel.
// EIG: one fission generation of the k-eigenvalue mode (DESIGN.md §3 C.14): the fission
// yield is nu / k of the running cycle, a child is born (id, group, direction) and then leaves through
// the census write-out instead of flying (in the last cycle it is only counted), and an inactive cycle
// scores nothing.  Also compiled out of the default kernel.
// IC: implicit capture with weight roulette (DESIGN.md §3 C.15): a collision multiplies the
// weight by (Sigma_s_row + Sigma_f)/Sigma_t and chooses among scattering and fission; below w_roulette the
// particle survives with probability w / w_survive.  Compiled out of the default kernel.
// DN: delayed neutrons (DESIGN.md §3 C.16): a new-born child is prompt or comes from a
// precursor group (then its time moves on by an exponential delay and its group comes from the delayed
// spectrum); a particle whose time is at or beyond the census time waits: census event of length 0, no
// score, time kept (also what a source particle of a source with a time extent does, C.17, until its
// birth time is reached).  Compiled out of the default kernel.
// MARCH: the tally mesh is finer than the lattice (configs 2 and 4, the eigenvalue pin cell, the dog-leg duct), so a
// flight scores several sub-segments and the warp-synchronous march waits for its longest flight.  When few lanes are
// still marching, their flights are suspended (24 bytes per slot) and regrouped 32 at a time in rounds of their own.
// CSG: the one lattice cell is divided into regions by quadric surfaces (DESIGN.md §3 C.18), which may
// move (C.19).  The region index travels in the ix field of the packed state; the cell's planes stay the outer box.
// MODE: how a flight scores the tally.  POOL_LEAN: the tally planes are the lattice planes and no cell holds a pin
// (configs 1, 3 and 5): one segment per flight, scored in the particle's own cell; the cylinder code is compiled out
// and the rare flight that starts exactly on a plane of its cell, heading out, marches alone in march_alone() — the
// hot loop carries neither the march's code nor its registers.  POOL_PLAIN: the general kernel (pins; any tally mesh,
// warp-synchronous march).  POOL_MARCH: POOL_PLAIN + suspended / regrouped marches.
enum { POOL_LEAN = 0, POOL_PLAIN = 1, POOL_MARCH = 2 };
template <bool TC, bool EIG, bool IC, bool DN, int MODE, bool CSG>
__global__ void __launch_bounds__(POOL_THREADS, MB_POOL)
k_pool(DevProblem P, TableLayout L, int use_smem, Bank Bin, Bank Bout, Ctl *ctl, Queues Q)
{
  constexpr bool MARCH = MODE == POOL_MARCH, LEAN = MODE == POOL_LEAN;
  // the regrouped-march variants call shared copies of the Philox block and of the divisions outside the march loop:
  // their hot code is just above the 32 KB instruction cache of an SM (profiles/pool_dogleg_r2.md: 1.6 warps per issue
  // wait for instructions); measured: dog-leg duct +3.4 %, config 2 +2.5 %; the plain general variants (larger still:
  // config 4 -2.5 %, eigenvalue pin cell -2 %) and the lean ones (which fit) inline everything
  constexpr bool PHX = MARCH;
  constexpr bool PHASE = MODE == POOL_PLAIN && !EIG;   // (eigenvalue pin cell: -1 %; regrouped march: -2 %; lean: -1 %)
  constexpr bool FASTPLANE = LEAN;      // (measured in the general variants too: config 4 +1 %, the others unchanged: left out there)
  static_assert(!(LEAN && CSG), "the CSG variants use the general kernel");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ unsigned long long s_cnt[N_CNT];
  // (the host takes this path only when the tables fit in shared memory: use_smem != 0)
  Tables T;
  {
    double *const tab = (double *)smem_raw;
    for (int i = threadIdx.x; i < L.total; i += blockDim.x) tab[i] = __ldg(P.xs4 + i);
    T.xs4 = tab + L.xs4; T.cdf_s = tab + L.cdf_s; T.cdf_chi = tab + L.cdf_chi;
    T.cdf_src = tab + L.cdf_src; T.speed = tab + L.speed;
  }
  // lattice plane tables: read by every flight
  double *const s_px = (double *)(smem_raw + pool_table_bytes(L, use_smem));
  double *const s_py = s_px + (P.nx + 1);
  double *const s_pz = s_py + (P.ny + 1);
  for (int i = threadIdx.x; i <= P.nx; i += blockDim.x) s_px[i] = __ldg(P.px + i);
  for (int i = threadIdx.x; i <= P.ny; i += blockDim.x) s_py[i] = __ldg(P.py + i);
  for (int i = threadIdx.x; i <= P.nz; i += blockDim.x) s_pz[i] = __ldg(P.pz + i);
  // leading zeros of a scatter CDF row (no up-scatter: the first g entries) can never be selected
  // (xi > 0): the search starts behind them
  uint8_t *const s_j0 = (uint8_t *)(s_pz + (P.nz + 1));
  for (int r = threadIdx.x; r < P.n_mat * P.G; r += blockDim.x) {
    int j = 0;
    while (j < P.G - 1 && !(__ldg(P.cdf_s + r * P.G + j) > 0.0)) ++j;
    s_j0[r] = (uint8_t)j;
  }
  // G <= 8: every scatter CDF row once more as eight fp32 thresholds (entries from G - 1 on: +inf), for the
  // first guess of the group-transfer search (A9 below)
  float *const s_cdf_f = (float *)(smem_raw + pool_table_bytes(L, use_smem) +
                                   ((((size_t)(P.nx + P.ny + P.nz + 3) * 8) + (size_t)P.n_mat * P.G + 15) & ~(size_t)15));
  if (LEAN && P.G <= 8)
    for (int i = threadIdx.x; i < P.n_mat * P.G * 8; i += blockDim.x) {
      const int r = i >> 3, j = i & 7;
      s_cdf_f[i] = j < P.G - 1 ? __double2float_rn(__ldg(P.cdf_s + r * P.G + j)) : __int_as_float(0x7F800000);
    }
  if (threadIdx.x < N_CNT) s_cnt[threadIdx.x] = 0ull;
  __syncthreads();

  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  // tally plane tables: staged for the variants that march (else read through the L1)
  double *const s_tx = (double *)(smem_raw + pool_table_bytes(L, use_smem) + pool_plane_bytes(P.nx, P.ny, P.nz, P.n_mat, P.G));
  double *const s_ty = s_tx + (P.tnx + 1), *const s_tz = s_ty + (P.tny + 1), *const s_tt = s_tz + (P.tnz + 1);
  if (MARCH) {
    for (int i = threadIdx.x; i <= P.tnx; i += blockDim.x) s_tx[i] = __ldg(P.tx + i);
    for (int i = threadIdx.x; i <= P.tny; i += blockDim.x) s_ty[i] = __ldg(P.ty + i);
    for (int i = threadIdx.x; i <= P.tnz; i += blockDim.x) s_tz[i] = __ldg(P.tz + i);
    for (int i = threadIdx.x; i <= P.tnt; i += blockDim.x) s_tt[i] = __ldg(P.tt + i);
    __syncthreads();
  }
  const double *const Tx = MARCH ? s_tx : P.tx, *const Ty = MARCH ? s_ty : P.ty, *const Tz = MARCH ? s_tz : P.tz,
               *const Tt = MARCH ? s_tt : P.tt;
  // quadric coefficients (CSG)
  double *const s_coef = (double *)(smem_raw + pool_table_bytes(L, use_smem) + pool_plane_bytes(P.nx, P.ny, P.nz, P.n_mat, P.G) +
                                    pool_tally_plane_bytes(P.tnx, P.tny, P.tnz, P.tnt, MARCH));
  if (CSG) {
    for (int i = threadIdx.x; i < P.csg_n_surf * 10; i += blockDim.x) s_coef[i] = __ldg(P.csg_coef + i);
    __syncthreads();
  }
  unsigned char *pool = smem_raw + pool_table_bytes(L, use_smem) + pool_plane_bytes(P.nx, P.ny, P.nz, P.n_mat, P.G) +
                        pool_tally_plane_bytes(P.tnx, P.tny, P.tnz, P.tnt, MARCH) + pool_csg_bytes(CSG ? P.csg_n_surf : 0) +
                        (size_t)wid * pool_bytes(MARCH);
  double2 *const s_xy = (double2 *)pool;
  double2 *const s_zt = s_xy + PW;
  double2 *const s_uxy = s_zt + PW;
  double2 *const s_uzw = s_uxy + PW;
  ulonglong2 *const s_idp = (ulonglong2 *)(s_uzw + PW);
  unsigned long long *const h_pid = (unsigned long long *)(s_idp + PW);   // hash ring: id, (ectr | event << 24)
  int *const s_mat = (int *)(h_pid + HRING);
  uint32_t *const h_ce = (uint32_t *)(s_mat + PW);
  uint8_t *const l_f = (uint8_t *)(h_ce + HRING);   // flight-ready
  uint8_t *const l_x = l_f + PW;                    // collision-ready and unborn children
  uint8_t *const l_z = l_x + PW;                    // waiting for the census write-out
  uint8_t *const l_free = l_z + PW;
  // suspended tally marches (MARCH): flight length, last crossing distance, tally indices; their list
  double *const s_md = (double *)(pool + POOL_BYTES);
  double *const s_ms = s_md + PW;
  unsigned long long *const s_mj = (unsigned long long *)(s_ms + PW);
  uint8_t *const l_m = (uint8_t *)(s_mj + PW);
  for (int i = lane; i < PW; i += 32) l_free[i] = (uint8_t)i;
  __syncwarp();
  uint32_t nF = 0, nX = 0, nZ = 0, nFree = PW, nH = 0, nM = 0;     // warp-uniform list lengths
  bool blocked = false;                             // the last collision round had to put fissions back

  const uint32_t n_end = ctl->n_active;             // active bank range [fetch, n_end)
  const uint32_t fetch_chunk = ctl->pool_chunk;
  // (spill_limit of the control block does not change during a launch: it is read in the spill path, which is rare,
  // instead of occupying a register of the hot loop)
  const double t_k = ctl->t_k;
  const unsigned long long seedb = ctl->seedb;
  const bool last_step = ctl->last_step != 0u;
  const double eig_k = EIG ? ctl->eig_k : 1.0;
  const bool score_on = !EIG || ctl->score != 0u;
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
  if (LEAN && P.simple_tally == 2) jt_step = -1;    // (tests, MCDC_LEAN=2: no flight takes the single-segment path, all march alone)
  // time-crossing block: the time bin whose upper edge is this step's census time (C.13)
  int jt_edge = -1;
  if (TC) {
    int lo = 0, hi = P.tnt;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(P.tt + mid) < t_k) lo = mid; else hi = mid; }
    if (__ldg(P.tt + lo + 1) == t_k) jt_edge = lo;
    else if (__ldg(P.tt + 1) == t_k) jt_edge = 0;
  }
  const double t_lo_step = jt_step >= 0 ? __ldg(P.tt + jt_step) : 0.0;
  const int g_stride = P.tnz * P.tny * P.tnx;
  if (!((long long)g_stride * G < (1ll << 30))) jt_step = -1;
  const long long bin_t0 = (long long)(jt_step >= 0 ? jt_step : 0) * G * g_stride;

  // Event counters.  Every lane adds its own events of a round into packed fields of three words (6 bits each, the
  // secondaries 8: a lane adds at most 1, or 7 children, per round); every 32nd round the fields are summed over the
  // warp and added to the warp's counters in shared memory, before a field can overflow.  (One warp reduction and
  // twelve unpacked uniform counters per round cost more instructions, and twelve registers of the hot loop.)
  //   accF: crossings | reflections << 6 | leaks << 12 | census << 18 | lost << 24      (flight rounds)
  //   accG: flights | single-segment scores << 6                                        (flight rounds)
  //   accX: collisions | scatters << 6 | captures << 12 | fissions << 18 | secondaries << 24
  __shared__ uint32_t s_wc[POOL_WARPS][12];
  if (threadIdx.x < POOL_WARPS * 12) (&s_wc[0][0])[threadIdx.x] = 0u;
  __syncthreads();
  uint32_t accF = 0, accG = 0, accX = 0;
  // (the general variants keep the per-round warp reduction into uniform counters: their rounds are long, and with
  // the packed words the regrouped-march kernel measured 2.6 % slower)
  uint32_t c_flights = 0, c_cross = 0, c_refl = 0, c_leak = 0, c_census = 0, c_lost = 0;
  uint32_t c_coll = 0, c_scat = 0, c_capt = 0, c_fis = 0, c_sec = 0;
  uint32_t c_segments = 0;                           // segments of tally marches (no bound per lane and round)
  unsigned long long fp = 0ull;
  auto counters_flush = [&]() {
    const uint32_t fe = __reduce_add_sync(0xffffffffu, accF & 0x0003F03Fu), fo = __reduce_add_sync(0xffffffffu, (accF >> 6) & 0x0003F03Fu),
                   ft = __reduce_add_sync(0xffffffffu, accF >> 24);
    const uint32_t xe = __reduce_add_sync(0xffffffffu, accX & 0x0003F03Fu), xo = __reduce_add_sync(0xffffffffu, (accX >> 6) & 0x0003F03Fu),
                   xt = __reduce_add_sync(0xffffffffu, accX >> 24);
    const uint32_t gg = __reduce_add_sync(0xffffffffu, (accG & 0x3Fu) | ((accG & 0xFC0u) << 6));
    if (lane == 0) {
      uint32_t *const w = s_wc[wid];
      w[0] += (gg & 0xFFFu) + c_flights; w[1] += (gg >> 12) + c_segments;                  // flights, segments
      w[2] += (fe & 0xFFFu) + c_cross; w[3] += (fo & 0xFFFu) + c_refl; w[4] += (fe >> 12) + c_leak;   // cross, refl, leak
      w[5] += (fo >> 12) + c_census; w[6] += ft + c_lost;                                  // census, lost
      w[7] += (xe & 0xFFFu) + c_coll; w[8] += (xo & 0xFFFu) + c_scat; w[9] += (xe >> 12) + c_capt;     // coll, scat, capt
      w[10] += (xo >> 12) + c_fis; w[11] += xt + c_sec;                                    // fis, sec
    }
    accF = 0u; accG = 0u; accX = 0u; c_segments = 0u;
    c_flights = c_cross = c_refl = c_leak = c_census = c_lost = c_coll = c_scat = c_capt = c_fis = c_sec = 0u;
  };

  uint32_t rng_next = 0, rng_end = 0, round = 0;
  bool exhausted = false;

  // terminal events wait in a ring; a round of kind "hash" takes 32 of them (so nH stays < HRING)
  auto ring_push = [&](bool has, uint64_t pid, uint32_t ectr, int ev) {
    const unsigned b = __ballot_sync(0xffffffffu, has);
    if (has) { const uint32_t k = nH + __popc(b & lt_mask); h_pid[k] = pid; h_ce[k] = ectr | ((uint32_t)ev << 24); }
    nH += __popc(b);
  };

  for (;;) {
    // (with a full round of flights ready, fewer than 32 census particles waiting and no fission put back, neither the
    // entry nor the exit nor the idle test below can apply: one test instead of all of theirs)
    if (nF < 32u || nZ >= 32u || blocked) {
    // ---- entry: deal reserved entries of the active bank to free pool slots ----
    if (nF < 32u && nFree > (uint32_t)POOL_RESERVE && !exhausted) {
      if (rng_next == rng_end) {
        // guided reservation: chunks shrink with what is left so that the warps finish together
        uint32_t b = 0, ch = 32u;
        if (lane == 0) {
          const uint32_t seen = ld_volatile_u32(&ctl->fetch);
          const uint32_t left = seen < n_end ? n_end - seen : 0u;
          ch = min(max(left / (2u * gridDim.x * POOL_WARPS), 32u), fetch_chunk);
          b = atomicAdd(&ctl->fetch, ch);
        }
        b = __shfl_sync(0xffffffffu, b, 0); ch = __shfl_sync(0xffffffffu, ch, 0);
        rng_next = min(b, n_end); rng_end = min(b + ch, n_end);
        if (rng_next == rng_end) exhausted = true;
      }
      if (!exhausted) {
        const uint32_t cnt = min(min(nFree - (uint32_t)POOL_RESERVE, 32u), rng_end - rng_next);
        bool unborn = false;
        uint32_t slot = 0;
        if ((uint32_t)lane < cnt) {
          slot = l_free[nFree - 1u - lane];
          const uint32_t i = rng_next + lane;
          const double2 a = Bin.xy[i], b2 = Bin.zt[i], c2 = Bin.uxy[i], e2 = Bin.uzw[i];
          ulonglong2 id = Bin.idp[i];
          const int cell = CSG ? 0 : (pk_iz(id.y) * P.ny + pk_iy(id.y)) * P.nx + pk_ix(id.y);
          const int pin = (!CSG && !LEAN && P.has_pins) ? (int)__ldg(P.mat_inner + cell) : -1;
          const int m = CSG ? (pk_ix(id.y) == CSG_NO_REGION ? 0 : (int)__ldg(P.csg_rmat + pk_ix(id.y)))
                            : (!LEAN && pk_inside(id.y)) ? pin : (int)__ldg(P.mat_outer + cell);
          int mm = mat_pack(m, pin);
          if (id.y & 1ull) {                         // an unborn child that a full pool handed to the bank
            unborn = true; id.y &= ~1ull;
            mm |= MAT_UNBORN | ((int)c2.x << 16);
          }
          s_xy[slot] = a; s_zt[slot] = b2; s_uxy[slot] = c2; s_uzw[slot] = e2; s_idp[slot] = id;
          s_mat[slot] = mm;
        }
        const unsigned bu = __ballot_sync(0xffffffffu, unborn);
        const unsigned bn = __ballot_sync(0xffffffffu, (uint32_t)lane < cnt && !unborn);
        if ((uint32_t)lane < cnt) {
          if (unborn) l_x[nX + __popc(bu & lt_mask)] = (uint8_t)slot;
          else l_f[nF + __popc(bn & lt_mask)] = (uint8_t)slot;
        }
        nFree -= cnt; nF += __popc(bn); nX += __popc(bu); rng_next += cnt;
        __syncwarp();
      }
    }
    // ---- exit: census write-out, 32 records per atomic ----
    if (nZ >= 32u || (nZ > 0u && ((nF == 0u && nX == 0u && nM == 0u) || blocked))) {
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
    if (nF == 0u && nX == 0u && nM == 0u && nH < 32u) {
      if (exhausted && nZ == 0u) break;
      continue;
    }
    }
    if ((round++ & 31u) == 31u) {
      if (LEAN) counters_flush();
      if ((round & 63u) == 0u) {                                                   // run is invalid: stop
        uint32_t ov = 0;
        if (lane == 0) ov = ld_volatile_u32(&ctl->overflow);
        if (__shfl_sync(0xffffffffu, ov, 0) != 0u) break;
      }
    }

    // one event kind per round: a full warp of one kind if there is one, else the longer list
    // (after a collision round that had to put fissions back, flights go first)
    int pick;                                         // 0 flight, 1 collision / birth, 2 hash, 3 resumed marches
    if (nH >= 32u) pick = 2;
    else if (MARCH && nM >= 32u) pick = 3;
    // (plain general variants: all warps of an SM lean towards the same kind of round — flights in even, collisions
    // in odd periods of 2^14 SM clocks — so that they run through the same code at about the same time: the code a
    // launch of config 4 executes is 38-45 KB, the instruction cache of an SM 32 KB, and 23 % of its stall samples
    // waited for instructions.  Config 4 +9 %; it changes the order of rounds only, no result.)
    else if (PHASE && !blocked && ((clock64() >> POOL_PHASE_SHIFT) & 1ll) == 0ll && nF >= (uint32_t)POOL_PHASE_MIN) pick = 0;
    else if (PHASE && !blocked && ((clock64() >> POOL_PHASE_SHIFT) & 1ll) != 0ll && nX >= (uint32_t)POOL_PHASE_MIN) pick = 1;
    else if (nX >= 32u && !blocked) pick = 1;
    else if (nF >= 32u) pick = 0;
    else if (blocked && nF) pick = 0;
    else if (MARCH && nM > 0u && nM >= max(nF, nX)) pick = 3;
    else pick = nX >= nF ? 1 : 0;

    // ---- the first Philox block of every kind of round is drawn here (one copy of the code) ----
    uint32_t cnt, slot = 0;
    bool active;
    uint64_t pid = 0, pk = 0;
    int mm = 0;
    uint32_t c0 = 0, c1 = 0, c2 = 0, c3 = 0;
    if (pick == 2) {
      cnt = 32u; active = true; nH -= 32u;
      const uint32_t ce = h_ce[nH + lane];
      pid = h_pid[nH + lane]; c0 = ce & 0xFFFFFFu; c1 = BLK_FINGERPRINT + (ce >> 24);
    } else {
      // idle lanes (there are few) repeat the work of lane 0 on its slot and are masked where it has
      // effects: the event code stays free of per-lane guards
      if (pick == 0) { cnt = min(nF, 32u); active = (uint32_t)lane < cnt; slot = l_f[nF - 1u - (active ? lane : 0)]; nF -= cnt; }
      else if (MARCH && pick == 3) { cnt = min(nM, 32u); active = (uint32_t)lane < cnt; slot = l_m[nM - 1u - (active ? lane : 0)]; nM -= cnt; }
      else { cnt = min(nX, 32u); active = (uint32_t)lane < cnt; slot = l_x[nX - 1u - (active ? lane : 0)]; nX -= cnt; }
      const ulonglong2 id = s_idp[slot];
      pid = id.x; pk = id.y; mm = s_mat[slot];
      c0 = pk_ectr(pk);
      c1 = pick == 0 ? (uint32_t)BLK_DCOL : ((mm & MAT_UNBORN) ? (uint32_t)BLK_CHILD + (uint32_t)((mm >> 16) & 7) : (uint32_t)BLK_REACT);
      c2 = (uint32_t)seedb; c3 = (uint32_t)(seedb >> 32);
    }
    // (a flight round draws its block further down, in one instruction stream with the plane distances,
    // which do not depend on it)
    U4 r1 = U4{0u, 0u, 0u, 0u};
    if (pick == 1 || pick == 2) r1 = philox_site<PHX>((uint32_t)pid, (uint32_t)(pid >> 32), c0, c1, c2, c3);
    if (pick == 2) {
      fp += ((unsigned long long)r1.x << 32) | (unsigned long long)r1.y;
      __syncwarp();
      continue;
    }

    if (pick == 0 || (MARCH && pick == 3)) {
      // ================= flight round (A3-A7, A11); with pick 3 the rest of suspended flights =================
      blocked = false;
      const bool resumed = MARCH && pick == 3;
      Lane p;
      {
        const double2 a = s_xy[slot], b2 = s_zt[slot], cc = s_uxy[slot], e2 = s_uzw[slot];
        p.x = a.x; p.y = a.y; p.z = b2.x; p.t = b2.y; p.ux = cc.x; p.uy = cc.y; p.uz = e2.x; p.w = e2.y;
        p.pid = 0; p.ectr = c0;
        p.g = pk_g(pk); p.ix = pk_ix(pk); p.iy = pk_iy(pk);
        p.iz = pk_iz(pk); p.inside = pk_inside(pk);
        p.m = mm & 0xFF; p.pin = ((mm >> 8) & 0xFF) - 1;
        // (lean variants: a particle that crossed a lattice plane in its last flight carries "material unknown"; the map
        // of the cell it entered is read here, where the load hides behind the Philox block and the plane distances)
        if (LEAN && p.m == MAT_UNKNOWN) p.m = (int)__ldg(P.mat_outer + (p.iz * P.ny + p.iy) * P.nx + p.ix);
      }
      bool dir_dirty = false;
      int outcome = 0;                  // 0 dead, 1 flight-ready, 2 collision, 3 census bank
      int end_ev = -1;
      uint32_t cw = 0;                   // cross | refl << 6 | leak << 12 | census << 18 | lost << 24
      const double v = T.speed[p.g];
      const int reg = p.ix;                            // CSG: the ix field holds the region, the box is cell 0
      int reg_out = reg;
      if (CSG) p.ix = 0;
      const double lx = s_px[p.ix], hx = s_px[p.ix + 1];
      const double ly = s_py[p.iy], hy = s_py[p.iy + 1];
      const double lz = s_pz[p.iz], hz = s_pz[p.iz + 1];
      double d = 0.0; int ev = 0, surf = 0;
      double tau_next = INF;                           // CSG: next break time of the surfaces' motion
      bool waiting = false, worn = false;
      if (!resumed) {
      // A3-A5 distances and event
      const double sig_t = T.xs4[(p.m * G + p.g) * 4];
      r1 = philox_site<PHX>((uint32_t)pid, (uint32_t)(pid >> 32), c0, c1, c2, c3);
      double d_s;
      if (FASTPLANE) d_s = nearest_plane(lx, hx, ly, hy, lz, hz, p.x, p.y, p.z, p.ux, p.uy, p.uz, P.planes_finite != 0, surf);
      double d_c = PHX ? div_shared(-mc_log(u52(r1.x, r1.y)), sig_t) : -mc_log(u52(r1.x, r1.y)) / sig_t;
      if (d_c < 0.0) d_c = 0.0;
      if (!FASTPLANE) {
        const double dsx = PHX ? ratio_shared((p.ux > 0.0 ? hx : lx) - p.x, p.ux) : plane_dist2(lx, hx, p.x, p.ux);
        const double dsy = PHX ? ratio_shared((p.uy > 0.0 ? hy : ly) - p.y, p.uy) : plane_dist2(ly, hy, p.y, p.uy);
        const double dsz = PHX ? ratio_shared((p.uz > 0.0 ? hz : lz) - p.z, p.uz) : plane_dist2(lz, hz, p.z, p.uz);
        d_s = dsx;
        if (dsy < d_s) { d_s = dsy; surf = 1; }
        if (dsz < d_s) { d_s = dsz; surf = 2; }
      }
      if (!LEAN && P.has_pins && p.pin >= 0) {
        const double cx = 0.5 * (lx + hx), cy = 0.5 * (ly + hy);
        const double dcy = cyl_dist(p.x, p.y, p.ux, p.uy, cx, cy,
                                    __ldg(P.radius + (p.iz * P.ny + p.iy) * P.nx + p.ix), p.inside);
        if (dcy < d_s) { d_s = dcy; surf = 3; }
      }
      double d_m = INF;
      if (CSG) {
        // C.18: the quadric surfaces of the region in the order of its list; a moving surface (C.19) is seen from its
        // own frame: position minus its displacement at the start of the flight, direction minus velocity / speed
        if (reg != CSG_NO_REGION) {
          for (int j = 0; j < 8; ++j) {
            const int e = (int)__ldg(P.csg_rsurf + reg * 8 + j);
            if (e == 0) break;
            const int sf = (e > 0 ? e : -e) - 1;
            double px = p.x, py = p.y, pz = p.z, wx = p.ux, wy = p.uy, wz = p.uz;
            if (P.mv_n_tau > 0) {
              double dd[3], vel[3];
              surf_motion(P, sf, p.t, dd, vel);
              px = p.x - dd[0]; py = p.y - dd[1]; pz = p.z - dd[2];
              wx = p.ux - vel[0] / v; wy = p.uy - vel[1] / v; wz = p.uz - vel[2] / v;
            }
            const double dq = quadric_dist(s_coef + sf * 10, e > 0 ? 1.0 : -1.0, px, py, pz, wx, wy, wz);
            if (dq < d_s) { d_s = dq; surf = 4 + j; }
          }
        }
        // C.19: the flight stops at the next break time of the surfaces' motion
        for (int j = P.mv_n_tau - 1; j >= 0; --j) { const double tj = __ldg(P.mv_tau + j); if (tj > p.t) tau_next = tj; }
        if (tau_next < INF) { d_m = (tau_next - p.t) * v; if (d_m < 0.0) d_m = 0.0; }
      }
      double d_t = (t_k - p.t) * v;
      if (d_t < 0.0) d_t = 0.0;
      d = d_c;
      if (d_s < d) { d = d_s; ev = 1; }
      if (d_t < d) { d = d_t; ev = 2; }
      if (CSG && d_m < d) { d = d_m; ev = 3; }
      waiting = DN && p.t >= t_k;                      // C.16: a precursor that has not emitted yet
      if (waiting) { d = 0.0; ev = 2; }
      // a flight counter at its 24-bit limit would repeat the random streams: the particle ends as lost (C.1)
      // (and a particle that is in no region of the CSG, C.18)
      worn = c0 == 0xFFFFFFu || (CSG && reg == CSG_NO_REGION);
      if (worn) d = 0.0;
      } else {
        d = s_md[slot]; ev = (mm >> 25) & 3; surf = (mm >> 27) & 3;
      }
      // A6 tally march (warp-synchronous; same two paths as k_flight)
      bool lost = false;
      bool generic = active && score_on && !waiting;
      bool susp = false;                               // MARCH: the rest of this lane's march waits for a round of its own
      int fx = p.ix, fy = p.iy, fz = p.iz;           // spatial tally bin the flight ends in
      if ((LEAN || P.simple_tally) && !resumed) {
        // (bitwise, not short-circuit: predicate logic instead of divergent branches)
        const bool okx = ((lx < p.x) & (p.x < hx)) | ((p.x == lx) & ((p.ux >= 0.0) | (p.ix == 0))) |
                         ((p.x == hx) & ((p.ux < 0.0) | (p.ix == P.nx - 1)));
        const bool oky = ((ly < p.y) & (p.y < hy)) | ((p.y == ly) & ((p.uy >= 0.0) | (p.iy == 0))) |
                         ((p.y == hy) & ((p.uy < 0.0) | (p.iy == P.ny - 1)));
        const bool okz = ((lz < p.z) & (p.z < hz)) | ((p.z == lz) & ((p.uz >= 0.0) | (p.iz == 0))) |
                         ((p.z == hz) & ((p.uz < 0.0) | (p.iz == P.nz - 1)));
        const bool simple = okx & oky & okz & (jt_step >= 0) & (p.t >= t_lo_step) & (p.t < t_k);
        if (simple) generic = false;
        const bool score = active && simple && d > 0.0 && score_on;
        const int bin32 = p.g * g_stride + (p.iz * P.tny + p.iy) * P.tnx + p.ix;     // (G * g_stride < 2^30: see jt_step)
        const unsigned bs = __ballot_sync(0xffffffffu, score);
        if (LEAN) accG += score ? 64u : 0u; else c_segments += __popc(bs);
        if (LEAN && !P.aggregate_tally) { if (score) atomicAdd(P.tally + bin_t0 + bin32, p.w * d); }    // (a large tally: one RED per lane)
        else if (bs) warp_tally_add(P.tally, score ? (long long)bin_t0 + (long long)bin32 : -1ll, p.w * d, P.aggregate_tally != 0);
      }
      if (LEAN) {
        if (__any_sync(0xffffffffu, generic)) {          // (rare: see MODE)
          uint32_t r = 0;
          if (generic) {
            int fxyz[3];
            const MarchTables mt = {P.tx, P.ty, P.tz, P.tt, P.tnx, P.tny, P.tnz, P.tnt, P.hx, P.hy, P.hz, P.ht, P.tally, P.tcross_off};
            r = march_alone<TC>(mt, G, p.x, p.y, p.z, p.t, p.ux, p.uy, p.uz, p.w, v, d, p.g, fxyz);
            fx = fxyz[0]; fy = fxyz[1]; fz = fxyz[2];
            lost = (r >> 31) != 0u;
          }
          c_segments += __reduce_add_sync(0xffffffffu, lost ? 0u : r);
        }
      } else if (__any_sync(0xffffffffu, generic)) {
        int jx = 0, jy = 0, jz = 0, jt = 0;
        double sx = INF, sy = INF, sz = INF, st = INF, s_prev = 0.0;
        bool marching = generic;
        uint32_t nseg = 0, n_it = 0;
        long long cur = 0;
        const int st_y = P.tnx, st_z = P.tny * P.tnx;
        const long long st_t = (long long)G * g_stride;
        if (generic) {
          if (!resumed) {
            jx = find_interval_any(Tx, P.tnx, p.x, p.ux, P.hx);
            jy = find_interval_any(Ty, P.tny, p.y, p.uy, P.hy);
            jz = find_interval_any(Tz, P.tnz, p.z, p.uz, P.hz);
            jt = find_interval_any(Tt, P.tnt, p.t, 1.0, P.ht);
          } else {
            // where the march stopped: its indices and last crossing distance; the next crossing of every axis
            // is recomputed from the flight origin, as in every step of the march (App. C.2)
            const unsigned long long mj = s_mj[slot];
            jx = (int)(mj & 0xFFFFu); jy = (int)((mj >> 16) & 0xFFFFu); jz = (int)((mj >> 32) & 0xFFFFu); jt = (int)(mj >> 48);
            s_prev = s_ms[slot];
          }
          sx = PHX ? ratio_shared(Tx[jx + (p.ux > 0.0 ? 1 : 0)] - p.x, p.ux) : plane_dist_any(Tx, jx, p.x, p.ux);
          sy = PHX ? ratio_shared(Ty[jy + (p.uy > 0.0 ? 1 : 0)] - p.y, p.uy) : plane_dist_any(Ty, jy, p.y, p.uy);
          sz = PHX ? ratio_shared(Tz[jz + (p.uz > 0.0 ? 1 : 0)] - p.z, p.uz) : plane_dist_any(Tz, jz, p.z, p.uz);
          st = (Tt[jt + 1] - p.t) * v; if (st < 0.0) st = 0.0;
          // bin of the current sub-segment, kept up to date by one add per crossing
          cur = ((((long long)jt * G + p.g) * P.tnz + jz) * P.tny + jy) * P.tnx + jx;
        }
        for (;;) {
          long long bin = -1, cbin = -1; double val = 0.0;
          if (marching) {
            int axis = 0; double s_min = sx;
            if (sy < s_min) { s_min = sy; axis = 1; }
            if (sz < s_min) { s_min = sz; axis = 2; }
            if (st < s_min) { s_min = st; axis = 3; }
            const bool cross = s_min < d;
            const double len = (cross ? s_min : d) - s_prev;
            if (len > 0.0) {
              bin = cur;
              val = p.w * len; ++nseg;
            }
            if (cross) {
              // ONE branch-free copy of the step for all four axes: lanes crossing different planes run it together.
              // The operands are selected; the arithmetic is the definition's (App. C.2): a spatial axis gets
              // (edge - p) / u, the time axis (edge - t) v, both clamped at 0, from the flight origin.
              const bool spatial = axis < 3;
              const double ua = axis == 0 ? p.ux : axis == 1 ? p.uy : p.uz;
              const double pa = axis == 0 ? p.x : axis == 1 ? p.y : p.z;
              const double *const Pa = axis == 0 ? Tx : axis == 1 ? Ty : axis == 2 ? Tz : Tt;
              const int na = axis == 0 ? P.tnx : axis == 1 ? P.tny : axis == 2 ? P.tnz : P.tnt;
              const int jo = axis == 0 ? jx : axis == 1 ? jy : axis == 2 ? jz : jt;
              const bool up = !spatial || ua > 0.0;
              const int ja = jo + (up ? 1 : -1);
              const bool out = ja < 0 || ja >= na;
              const double edge = Pa[out ? 0 : ja + (up ? 1 : 0)];
              double sa = spatial ? (edge - pa) / ua : (edge - p.t) * v;
              if (sa < 0.0) sa = 0.0;
              if (out) { lost = true; sa = INF; }
              // the time passes the upper edge of time bin jt: time-crossing score (C.13)
              if (TC && !spatial) cbin = P.tcross_off + cur;
              cur += axis == 0 ? (long long)(up ? 1 : -1) : axis == 1 ? (long long)(up ? st_y : -st_y)
                   : axis == 2 ? (long long)(up ? st_z : -st_z) : st_t;
              jx = axis == 0 ? ja : jx; jy = axis == 1 ? ja : jy; jz = axis == 2 ? ja : jz; jt = axis == 3 ? ja : jt;
              sx = axis == 0 ? sa : sx; sy = axis == 1 ? sa : sy; sz = axis == 2 ? sa : sz; st = axis == 3 ? sa : st;
              s_prev = s_min;
              if (lost) marching = false;
            } else marching = false;
          }
          if (TC && __any_sync(0xffffffffu, cbin >= 0)) warp_tally_add(P.tally, cbin, p.w * v, P.aggregate_tally != 0);
          if (!__any_sync(0xffffffffu, bin >= 0 || marching)) break;
          if (__any_sync(0xffffffffu, bin >= 0)) warp_tally_add(P.tally, bin, val, P.aggregate_tally != 0);
          if (MARCH) {
            // few lanes left marching: suspend them (a round of resumed marches that started with few lanes, or has
            // run only a few iterations, goes on: every suspension must be paid for by progress)
            ++n_it;
            const uint32_t nm = (uint32_t)__popc(__ballot_sync(0xffffffffu, marching));
            if (nm > 0u && nm < (uint32_t)P.march_min && (resumed ? (cnt >= (uint32_t)P.march_min && n_it >= (uint32_t)P.march_iter_min) : n_it >= (uint32_t)P.march_first)) {
              susp = marching;
              break;
            }
          }
        }
        if (generic) { fx = jx; fy = jy; fz = jz; }
        c_segments += __reduce_add_sync(0xffffffffu, lost ? 0u : nseg);
        if (MARCH) {
          const unsigned bsu = __ballot_sync(0xffffffffu, susp);
          if (susp) {
            s_md[slot] = d; s_ms[slot] = s_prev;
            s_mj[slot] = (unsigned long long)(uint32_t)jx | ((unsigned long long)(uint32_t)jy << 16) |
                         ((unsigned long long)(uint32_t)jz << 32) | ((unsigned long long)(uint32_t)jt << 48);
            s_mat[slot] = (mm & 0x1FFFFFF) | (ev << 25) | (surf << 27);
            l_m[nM + __popc(bsu & lt_mask)] = (uint8_t)slot;
          }
          nM += __popc(bsu);
        }
      }
      // the lanes whose flight is complete: move, snap, dispatch (suspended flights keep their origin)
      const bool fin = active && !susp;
      if (LEAN) accG += fin ? 1u : 0u; else c_flights += (uint32_t)__popc(__ballot_sync(0xffffffffu, fin));
      // move, snap, dispatch
      const uint32_t end_ectr = p.ectr;
      lost = lost || worn;
      if (lost) { cw = 1u << 24; end_ev = END_LOST; }
      else {
        p.x = fma(d, p.ux, p.x); p.y = fma(d, p.uy, p.y); p.z = fma(d, p.uz, p.z);
        p.t = p.t + (PHX ? div_shared(d, v) : d / v);
        if (ev == 2) {                                   // A11 census
          if (!waiting) p.t = t_k;
          cw = 1u << 18; end_ev = END_CENSUS;
          ++p.ectr; outcome = last_step ? 0 : 3;
        } else if (CSG && ev == 3) {                     // C.19 break time: nothing else happens
          p.t = tau_next; cw = 1u; ++p.ectr; outcome = 1;
        } else if (CSG && ev == 1 && surf >= 4) {        // C.18 quadric surface: the region on its other side
          const int e = (int)__ldg(P.csg_rsurf + reg * 8 + (surf - 4));
          const int nr = find_region(P, s_coef, reg, (e > 0 ? e : -e) - 1, p.x, p.y, p.z, p.t);
          reg_out = nr < 0 ? CSG_NO_REGION : nr;
          p.m = nr < 0 ? 0 : (int)__ldg(P.csg_rmat + nr);
          cw = 1u; ++p.ectr; outcome = 1;
        } else if (ev == 1) {                            // A7 surface
          outcome = 1;
          if (!LEAN && surf == 3) {
            p.inside ^= 1;
            p.m = p.inside ? p.pin : (int)__ldg(P.mat_outer + (p.iz * P.ny + p.iy) * P.nx + p.ix);
            cw = 1u; ++p.ectr;
          } else {
            const double u = surf == 0 ? p.ux : surf == 1 ? p.uy : p.uz;
            const bool up = u > 0.0;
            const int idx = surf == 0 ? p.ix : surf == 1 ? p.iy : p.iz;
            const int nax = surf == 0 ? P.nx : surf == 1 ? P.ny : P.nz;
            const double edge = surf == 0 ? (up ? hx : lx) : surf == 1 ? (up ? hy : ly) : (up ? hz : lz);
            if (surf == 0) p.x = edge; else if (surf == 1) p.y = edge; else p.z = edge;
            const bool outer = up ? (idx == nax - 1) : (idx == 0);
            if (!outer) {
              const int ni = idx + (up ? 1 : -1);
              if (surf == 0) p.ix = ni; else if (surf == 1) p.iy = ni; else p.iz = ni;
              if (LEAN) { p.inside = 0; p.m = MAT_UNKNOWN; cw = 1u; ++p.ectr; }
              else { p.inside = 0; lane_material(P, p); cw = 1u; ++p.ectr; }
            } else if (P.bc[2 * surf + (up ? 1 : 0)] == 1) {
              if (surf == 0) p.ux = -p.ux; else if (surf == 1) p.uy = -p.uy; else p.uz = -p.uz;
              dir_dirty = true; cw = 1u << 6; ++p.ectr;
            } else { cw = 1u << 12; end_ev = END_LEAK; outcome = 0; }
          }
        } else outcome = 2;                              // collision: a later round of that kind
      }
      if (TC) {                                              // alive at the census time, a tally time edge (C.13)
        const bool sc = fin && !lost && ev == 2 && jt_edge >= 0 && !waiting;
        if (LEAN && !P.aggregate_tally) {                    // (a large tally: one RED per lane, 32-bit bin arithmetic)
          if (sc) atomicAdd(P.tally + (P.tcross_off + (long long)jt_edge * G * g_stride) + (p.g * g_stride + (fz * P.tny + fy) * P.tnx + fx), p.w * v);
        } else {
          const long long cb = sc ? P.tcross_off + ((((long long)jt_edge * G + p.g) * P.tnz + fz) * P.tny + fy) * P.tnx + fx : -1ll;
          if (__any_sync(0xffffffffu, sc)) warp_tally_add(P.tally, cb, p.w * v, P.aggregate_tally != 0);
        }
      }
      if (LEAN) accF += fin ? cw : 0u;
      else {
        const uint32_t sw = __reduce_add_sync(0xffffffffu, fin ? cw : 0u);
        c_cross += sw & 63u; c_refl += (sw >> 6) & 63u; c_leak += (sw >> 12) & 63u;
        c_census += (sw >> 18) & 63u; c_lost += (sw >> 24) & 63u;
      }
      ring_push(fin && end_ev >= 0, LEAN ? pid : s_idp[slot].x, end_ectr, end_ev);
      // back to the pool, onto the list of the next event
      if (fin && outcome != 0) {
        s_xy[slot] = make_double2(p.x, p.y);
        s_zt[slot] = make_double2(p.z, p.t);
        if (dir_dirty) { s_uxy[slot] = make_double2(p.ux, p.uy); s_uzw[slot] = make_double2(p.uz, p.w); }
        s_idp[slot].y = pack_state(p.ectr, p.g, CSG ? reg_out : p.ix, p.iy, p.iz, p.inside);
        s_mat[slot] = mat_pack(p.m, p.pin);
      }
      const unsigned b1 = __ballot_sync(0xffffffffu, fin && outcome == 1);
      const unsigned b2 = __ballot_sync(0xffffffffu, fin && outcome == 2);
      const unsigned b3 = __ballot_sync(0xffffffffu, fin && outcome == 3);
      const unsigned b0 = __ballot_sync(0xffffffffu, fin && outcome == 0);
      if (fin) {
        if (outcome == 1) l_f[nF + __popc(b1 & lt_mask)] = (uint8_t)slot;
        else if (outcome == 2) l_x[nX + __popc(b2 & lt_mask)] = (uint8_t)slot;
        else if (outcome == 3) l_z[nZ + __popc(b3 & lt_mask)] = (uint8_t)slot;
        else l_free[nFree + __popc(b0 & lt_mask)] = (uint8_t)slot;
      }
      nF += __popc(b1); nX += __popc(b2); nZ += __popc(b3); nFree += __popc(b0);
      __syncwarp();
    } else {
      // ================= collision / birth round (A8-A10) =================
      // kind: 0 capture, 1 scatter, 2 fission, 3 fission put back, 4 birth of a fission child, 5 idle lane
      int kind = 0, g2 = 0;
      const int m = mm & 0xFF, g = pk_g(pk);
      const uint32_t ectr = c0;
      uint32_t n_out = 0, n_new = 0;
      double w = s_uzw[slot].y;
      const double *xs = T.xs4 + (m * G + g) * 4;
      const double sig_t = xs[0], ssr = xs[1], sf = xs[2], nu = EIG ? xs[3] / eig_k : xs[3];
      uint64_t key2 = pid; uint32_t e2c = ectr, blk2 = BLK_FIS_N;
      int dn_j = -1;                                    // precursor group of a delayed child being born
      bool ic_kill = false, ic_scatter = false;
      if (IC) {
        // C.15: the capture is taken out of the weight; then the roulette; then scatter | fission
        // (all lanes pass here together: the warp-wide vote must not sit in the divergent branch below)
        const bool coll = !(mm & MAT_UNBORN);
        const double surv = ssr + sf;
        ic_kill = coll && !(surv > 0.0);
        if (coll && !ic_kill) w = w * (surv / sig_t);
        const bool play = active && coll && !ic_kill && w < P.ic_w_roulette;
        if (__any_sync(0xffffffffu, play)) {
          const U4 rr = philox_site<PHX>((uint32_t)pid, (uint32_t)(pid >> 32), ectr, BLK_ROULETTE, (uint32_t)seedb, (uint32_t)(seedb >> 32));
          if (play) { if (u52(rr.x, rr.y) * P.ic_w_survive < w) w = P.ic_w_survive; else ic_kill = true; }
        }
        ic_scatter = !(sf > 0.0);
      }
      if (mm & MAT_UNBORN) {
        kind = 4;
        key2 = (1ull << 63) | ((((uint64_t)r1.x << 32) | (uint64_t)r1.y) >> 1);   // the child's id (C.1)
        e2c = 0u; blk2 = BLK_SRC_ZG;
      } else {
        const double a = u52(r1.x, r1.y) * (IC ? ssr + sf : sig_t);
        if (IC && ic_kill) kind = 0;
        else if (a < ssr || (IC && ic_scatter)) {
          kind = 1;
          const double *row = T.cdf_s + (m * G + g) * G;
          const double xi = u52(r1.z, r1.w);
          // A9 group transfer: the first entry of the row's CDF above xi (C.3).  Lean variants, G <= 8: a first guess comes from
          // eight fp32 copies of the row (count of thresholds <= xi, no loop, no divergence); it is the answer exactly
          // when the fp64 row confirms it (entry above xi, entry before it not), which a row that does not decrease
          // makes unique; else, and for larger G, the linear search of the definition.  (The general variants keep the
          // search alone: with the guess the regrouped-march kernel measured 4.7 % slower.)
          bool found = false;
          if (LEAN && G <= 8) {
            const float xf = __double2float_rn(xi);
            const float4 fa = *(const float4 *)(s_cdf_f + (m * G + g) * 8), fb = *(const float4 *)(s_cdf_f + (m * G + g) * 8 + 4);
            const int c = (xf >= fa.x) + (xf >= fa.y) + (xf >= fa.z) + (xf >= fa.w) + (xf >= fb.x) + (xf >= fb.y) + (xf >= fb.z);
            found = (c == G - 1 || xi < row[c]) && (c == 0 || !(xi < row[c - 1]));
            g2 = c;
          }
          if (!found) {
            g2 = s_j0[m * G + g];
            while (g2 < G - 1 && !(xi < row[g2])) ++g2;
          }
        }
        else if (a < ssr + sf) kind = 2;
      }
      if (!active) kind = 5;
      // second block: number of children (fission) / group of the child (birth); third block: new direction
      // (scatter: the particle's stream; birth: the child's own stream).  Their inputs are known together, so
      // the two chains are drawn in one interleaved instruction stream (nearly every round needs both).
      U4 r2, r3;
      {
        const uint64_t key3 = kind == 4 ? key2 : pid;
        if (PHX) {
          r2 = philox_shared((uint32_t)key2, (uint32_t)(key2 >> 32), e2c, blk2, (uint32_t)seedb, (uint32_t)(seedb >> 32));
          r3 = philox_shared((uint32_t)key3, (uint32_t)(key3 >> 32), kind == 4 ? 0u : ectr,
                             kind == 4 ? (uint32_t)BLK_SRC_DIR : (uint32_t)BLK_SCAT_DIR, (uint32_t)seedb, (uint32_t)(seedb >> 32));
        } else
        philox4x32_10_x2((uint32_t)key2, (uint32_t)(key2 >> 32), e2c, blk2, (uint32_t)seedb, (uint32_t)(seedb >> 32),
                         (uint32_t)key3, (uint32_t)(key3 >> 32), kind == 4 ? 0u : ectr,
                         kind == 4 ? (uint32_t)BLK_SRC_DIR : (uint32_t)BLK_SCAT_DIR, (uint32_t)seedb, (uint32_t)(seedb >> 32),
                         r2, r3);
      }
      if (__any_sync(0xffffffffu, kind == 2 || kind == 4)) {
        if (kind == 2) { n_out = (uint32_t)(int)(nu + u52(r2.x, r2.y)); n_new = n_out > 0 ? n_out - 1 : 0; }
        else if (kind == 4) {
          const double *cdf_g = T.cdf_chi + m * G;
          if (DN && P.dn_J > 0) {
            // C.16: prompt with probability nu_p / nu, else from precursor group jd (g = the parent's group)
            const int J = P.dn_J;
            const double a_t = u52(r2.x, r2.y) * xs[3];
            double run = __ldg(P.dn_nup + m * G + g);
            if (!(a_t < run)) {
              dn_j = J - 1;
              for (int jj = 0; jj < J; ++jj) {
                run = run + __ldg(P.dn_nu + (m * G + g) * J + jj);
                if (a_t < run) { dn_j = jj; break; }
              }
              cdf_g = P.dn_cdf + (m * J + dn_j) * G;
            }
          }
          g2 = sample_cdf(cdf_g, G, u52(r2.z, r2.w));
        }
        if (DN && __any_sync(0xffffffffu, dn_j >= 0)) {      // emission delay from the child's own stream
          const U4 rd = philox_site<PHX>((uint32_t)key2, (uint32_t)(key2 >> 32), 0u, BLK_DELAY, (uint32_t)seedb, (uint32_t)(seedb >> 32));
          if (dn_j >= 0) {
            double2 zt = s_zt[slot];
            zt.y = zt.y + (-mc_log(u52(rd.x, rd.y))) / __ldg(P.dn_lambda + m * P.dn_J + dn_j);
            s_zt[slot] = zt;
          }
        }
      }
      if (__any_sync(0xffffffffu, kind == 1 || kind == 4)) {
        double ux, uy, uz;
        isotropic_dir(u52(r3.x, r3.y), u52(r3.z, r3.w), ux, uy, uz);
        if (kind == 1) {
          s_uxy[slot] = make_double2(ux, uy);
          s_uzw[slot] = make_double2(uz, w);
          uint64_t q = (pk & ~(0xFFull << 32)) | ((uint64_t)(uint32_t)g2 << 32);
          q = (q & 0x000000FFFFFFFFFFull) | ((uint64_t)(ectr + 1u) << 40);
          s_idp[slot] = make_ulonglong2(pid, q);
        } else if (kind == 4) {
          s_uxy[slot] = make_double2(ux, uy);
          s_uzw[slot] = make_double2(uz, w);
          s_idp[slot] = make_ulonglong2(key2, (pk & 0x00000000FFFFFFFFull) | ((uint64_t)(uint32_t)g2 << 32));
          s_mat[slot] = mm & 0xFFFF;
        }
      }
      // slots of particles that ended are free before the children ask for room
      // (a child born in the last generation of the eigenvalue mode is counted, not banked)
      const bool dies = kind == 0 || (kind == 2 && n_out == 0u) || (EIG && kind == 4 && last_step);
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
        const bool defer = n_new > 0u && incl > nFree;       // the family does not fit (in lane order)
        const unsigned bdef = __ballot_sync(0xffffffffu, defer);
        if (bdef) {
          const bool stuck = bdef == __ballot_sync(0xffffffffu, active) && nF == 0u;
          if (!stuck) {
            // put back: the same collision is drawn again later from the same counters
            if (defer) { kind = 3; l_x[nX + __popc(bdef & lt_mask)] = (uint8_t)slot; n_new = 0; }
            nX += __popc(bdef); blocked = true;
          } else {
            // a pool full of fission parents: their further children go, unborn, behind the active range
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
            if (spill_base + n_spill > ld_volatile_u32(&ctl->spill_limit)) { if (lane == 0) atomicExch(&ctl->overflow, 1u); spill_base = 0xFFFFFFFFu; }
            if (defer && spill_base != 0xFFFFFFFFu) {
              const double2 a2 = s_xy[slot], b2 = s_zt[slot];
              for (uint32_t j = 1; j < n_out; ++j) {
                const uint32_t o = spill_base + (isp - n_new) + (j - 1u);
                Bin.xy[o] = a2; Bin.zt[o] = b2;
                Bin.uxy[o] = make_double2((double)j, 0.0);
                Bin.uzw[o] = make_double2(0.0, w);
                Bin.idp[o] = make_ulonglong2(pid, pk | 1ull);
              }
            }
            if (defer) n_new = 0;                            // (their first child still takes the parent's slot)
          }
        }
        // families that fit: unborn children (parent id, flight counter and child index) into free slots
        // (their ranks are the prefix sums above unless a family was put back or spilled)
        uint32_t ifit = incl;
        if (bdef) {
          ifit = n_new;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, ifit, o);
            if (lane >= o) ifit += t;
          }
        }
        const uint32_t take = __shfl_sync(0xffffffffu, ifit, 31);
        if (n_new) {
          const double2 a2 = s_xy[slot], b2 = s_zt[slot];
          const int mb = (mm & 0xFFFF) | MAT_UNBORN;
          for (uint32_t j = 1; j <= n_new; ++j) {
            const uint32_t cs = l_free[nFree - 1u - (ifit - n_new + j - 1u)];
            s_xy[cs] = a2; s_zt[cs] = b2; s_uzw[cs] = make_double2(0.0, w);
            s_idp[cs] = make_ulonglong2(pid, pk);
            s_mat[cs] = mb | (int)(j << 16);
          }
        }
        __syncwarp();
        for (uint32_t k = lane; k < take; k += 32) l_x[nX + k] = l_free[nFree - 1u - k];
        nX += take; nFree -= take;
      }
      const bool flies = kind == 1 || (!EIG && kind == 4), born = kind == 2 && n_out > 0u;
      const unsigned b1 = __ballot_sync(0xffffffffu, flies);
      const unsigned b2 = __ballot_sync(0xffffffffu, born);
      if (EIG) {                                             // C.14: the new-born child is the next generation's
        const unsigned b4 = __ballot_sync(0xffffffffu, kind == 4);
        const unsigned bz = last_step ? 0u : b4;
        if (kind == 4 && !last_step) l_z[nZ + __popc(bz & lt_mask)] = (uint8_t)slot;
        nZ += __popc(bz); if (LEAN) accF += kind == 4 ? 1u << 18 : 0u; else c_census += __popc(b4);
      }
      if (flies) l_f[nF + __popc(b1 & lt_mask)] = (uint8_t)slot;
      if (born) {                                          // child 0 in the parent's slot
        l_x[nX + __popc(b2 & lt_mask)] = (uint8_t)slot; s_mat[slot] = (mm & 0xFFFF) | MAT_UNBORN;
        if (IC) s_uzw[slot].y = w;                         // (a fission put back keeps the old weight: it is drawn again)
      }
      nF += __popc(b1); nX += __popc(b2);
      // collisions | scatters << 6 | captures << 12 | fissions << 18 | secondaries << 24
      {
        uint32_t cw = 0;
        if (kind < 3) cw = 1u | (kind == 1 ? 1u << 6 : kind == 0 ? 1u << 12 : (1u << 18) | (n_out << 24));
        if (LEAN) accX += cw;
        else {
          const uint32_t sw = __reduce_add_sync(0xffffffffu, cw);
          c_coll += sw & 63u; c_scat += (sw >> 6) & 63u; c_capt += (sw >> 12) & 63u;
          c_fis += (sw >> 18) & 63u; c_sec += sw >> 24;
        }
      }
      if (EIG) ring_push(kind == 0 || kind == 2 || kind == 4, kind == 4 ? key2 : pid, kind == 4 ? 0u : ectr,
                         kind == 0 ? END_CAPTURE : kind == 2 ? END_FISSION : END_CENSUS);
      else ring_push(kind == 0 || kind == 2, pid, ectr, kind == 0 ? END_CAPTURE : END_FISSION);
      __syncwarp();
    }
  }
  if ((uint32_t)lane < nH) fp += end_hash(h_pid[lane], h_ce[lane] & 0xFFFFFFu, (int)(h_ce[lane] >> 24));

  counters_flush();
  if (lane == 0) {
    const int ks[12] = {K_FLIGHTS, K_SEGMENTS, K_CROSSINGS, K_REFLECTIONS, K_LEAKS, K_CENSUS, K_LOST,
                        K_COLLISIONS, K_SCATTERS, K_CAPTURES, K_FISSIONS, K_SECONDARIES};
#pragma unroll
    for (int i = 0; i < 12; ++i) { const uint32_t c = s_wc[wid][i]; if (c) atomicAdd(&s_cnt[ks[i]], (unsigned long long)c); }
  }
  warp_count64(s_cnt, K_FINGERPRINT, fp);
  flush_counts(s_cnt, ctl->cnt);
}

// after a pool launch: fission children that found the pools full sit behind the processed range
// (the spill window [spill_lo, bank_tail)); they become the next range, and the next spill window is
// the larger free part of the bank beside it
static __device__ __forceinline__ uint32_t pool_chunk_for(uint32_t n, uint32_t grid)
{
  return (unsigned long long)n > (unsigned long long)grid * POOL_WARPS * 512ull ? 128u : 32u;
}
__global__ void k_pool_begin(Ctl *ctl, uint32_t capacity, uint32_t grid)
{
  ctl->fetch = 0u; ctl->bank_tail = ctl->n_active; ctl->spill_lo = ctl->n_active; ctl->spill_limit = capacity;
  ctl->pool_chunk = pool_chunk_for(ctl->n_active, grid);
}
// waited != 0: the host reads the mirror and relaunches over the spilled children; else it has queued the rest
// of the batch already, and children left behind make the batch invalid (it is then run again, waiting)
__global__ void k_pool_next(Ctl *ctl, uint32_t *mirror, uint32_t capacity, uint32_t grid, uint32_t waited)
{
  const uint32_t lo = ctl->spill_lo, hi = ctl->overflow ? lo : ctl->bank_tail;
  ctl->fetch = lo;
  ctl->n_active = hi;
  ctl->pool_chunk = pool_chunk_for(hi - lo, grid);
  if (!waited && hi > lo) ctl->spill_seen = 1u;
  // everything outside [lo, hi) is free now: the next window is the larger side
  if (capacity - hi >= lo) { ctl->spill_lo = hi; ctl->bank_tail = hi; ctl->spill_limit = capacity; }
  else { ctl->spill_lo = 0u; ctl->bank_tail = 0u; ctl->spill_limit = lo; }
  ctl->iter += 1u;
  mirror[0] = hi - lo; mirror[1] = ctl->n_census; mirror[2] = ctl->overflow; mirror[3] = hi;
  mirror[4] = (uint32_t)ctl->cnt[K_FLIGHTS]; mirror[5] = (uint32_t)(ctl->cnt[K_FLIGHTS] >> 32);
}

}  // namespace mcdc
