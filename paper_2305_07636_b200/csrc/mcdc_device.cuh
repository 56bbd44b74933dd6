// mcdc_device.cuh — device-side building blocks of the event-based transport path
// (sm_100a).  Written independently of oracle/: no shared code, tables or headers.
// Definitions follow DESIGN.md §3 (C.1 RNG, C.2/App. B math, App. C geometry).
// Compiled with -fmad=false: every fused multiply-add below is an explicit fma().
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mcdc {

// ---------------------------------------------------------------- RNG (A2, C.1)
struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(uint32_t k0, uint32_t k1, uint32_t c0, uint32_t c1,
                                            uint32_t c2, uint32_t c3)
{
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = __umulhi(M0, c0), l0 = M0 * c0;
    const uint32_t h1 = __umulhi(M1, c2), l1 = M1 * c2;
    c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    k0 += W0; k1 += W1;
  }
  return U4{c0, c1, c2, c3};
}

// two independent blocks in one instruction stream: their rounds interleave, so each chain's multiply
// latency hides behind the other's (the collision round needs two blocks whose inputs are known together)
__device__ __forceinline__ void philox4x32_10_x2(uint32_t ka0, uint32_t ka1, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                                 uint32_t kb0, uint32_t kb1, uint32_t b0, uint32_t b1, uint32_t b2, uint32_t b3,
                                                 U4 &ra, U4 &rb)
{
  constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t ah0 = __umulhi(M0, a0), al0 = M0 * a0, ah1 = __umulhi(M1, a2), al1 = M1 * a2;
    const uint32_t bh0 = __umulhi(M0, b0), bl0 = M0 * b0, bh1 = __umulhi(M1, b2), bl1 = M1 * b2;
    a0 = ah1 ^ a1 ^ ka0; a1 = al1; a2 = ah0 ^ a3 ^ ka1; a3 = al0;
    b0 = bh1 ^ b1 ^ kb0; b1 = bl1; b2 = bh0 ^ b3 ^ kb1; b3 = bl0;
    ka0 += W0; ka1 += W1; kb0 += W0; kb1 += W1;
  }
  ra = U4{a0, a1, a2, a3}; rb = U4{b0, b1, b2, b3};
}

// purpose codes of the counter's second word
enum : uint32_t { BLK_SRC_XY = 0, BLK_SRC_ZG = 1, BLK_SRC_DIR = 2, BLK_SRC_PIN = 3, BLK_DCOL = 4,
                  BLK_REACT = 5, BLK_SCAT_DIR = 6, BLK_FIS_N = 7, BLK_ROULETTE = 8, BLK_DELAY = 9, BLK_SRC_TIME = 10, BLK_CHILD = 0x100,
                  BLK_FINGERPRINT = 0x200 };

__device__ __forceinline__ U4 draw_block(uint64_t pid, uint32_t ectr, uint32_t blk, uint64_t seedb)
{
  return philox4x32_10((uint32_t)pid, (uint32_t)(pid >> 32), ectr, blk, (uint32_t)seedb,
                       (uint32_t)(seedb >> 32));
}

// 52-bit uniform in (0,1): (k + 1/2) 2^-52, exact
__device__ __forceinline__ double u52(uint32_t hi, uint32_t lo)
{
  // k in the mantissa of a double in [1,2): 1 + k 2^-52; minus 1 and plus 2^-53 are both exact
  // ((2k+1) 2^-53 has at most 53 significant bits), so this is (k + 1/2) 2^-52 without a conversion
  // (the two words of that double directly: high = exponent | top 20 bits of hi, low = the 32 bits of (hi:lo) from bit 12)
  return (__hiloint2double((int)(0x3FF00000u | (hi >> 12)), (int)__funnelshift_r(lo, hi, 12)) - 1.0) + 1.1102230246251565404236316680908203125e-16;
}

// ------------------------------------------------------- math (C.2, App. B)
// Series coefficients live in constant memory: an fma then takes them as a constant-bank operand
// instead of two register moves per 64-bit immediate.  Each is ONE correctly rounded divide (App. B).
__constant__ double MC_LOG_C[11] = {1.0, 1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0, 1.0 / 13.0,
                                    1.0 / 15.0, 1.0 / 17.0, 1.0 / 19.0, 1.0 / 21.0};
__constant__ double MC_SIN_C[8] = {1.0, -1.0 / 6.0, 1.0 / 120.0, -1.0 / 5040.0, 1.0 / 362880.0, -1.0 / 39916800.0,
                                   1.0 / 6227020800.0, -1.0 / 1307674368000.0};
__constant__ double MC_COS_C[9] = {1.0, -1.0 / 2.0, 1.0 / 24.0, -1.0 / 720.0, 1.0 / 40320.0, -1.0 / 3628800.0,
                                   1.0 / 479001600.0, -1.0 / 87178291200.0, 1.0 / 20922789888000.0};
// log on (0,1], atanh series in s = f/(2+f), 11 terms, Horner with fma
__device__ __forceinline__ double mc_log(double x)
{
  const long long b = __double_as_longlong(x);
  int e = (int)((b >> 52) & 0x7FF) - 1023;
  double m = __longlong_as_double((b & 0x000FFFFFFFFFFFFFll) | 0x3FF0000000000000ll);
  if (m > 1.4142135623730951454746218587388284504413604736328125) { m *= 0.5; e += 1; }
  const double f = m - 1.0;
  const double s = f / (2.0 + f);
  const double z = s * s;
  double p = MC_LOG_C[10];
#pragma unroll
  for (int n = 9; n >= 0; --n) p = fma(p, z, MC_LOG_C[n]);
  return fma((double)e, 0.693147180559945286226763982995180413126945495605468750, (s + s) * p);
}

// cos(2 pi u), sin(2 pi u) for u in (0,1): octant reduction, Taylor with fma
__device__ __forceinline__ void mc_sincos2pi(double u, double &c, double &s)
{
  const double q4 = 4.0 * u;
  const int k = (int)q4;
  double r = q4 - (double)k;
  const bool swp = r > 0.5;
  if (swp) r = 1.0 - r;
  const double th = r * 1.5707963267948965579989817342720925807952880859375;
  const double z = th * th;
  double S = MC_SIN_C[7];                       // -1/15!
#pragma unroll
  for (int n = 6; n >= 0; --n) S = fma(S, z, MC_SIN_C[n]);
  S = th * S;
  double C = MC_COS_C[8];                       // +1/16!
#pragma unroll
  for (int n = 7; n >= 0; --n) C = fma(C, z, MC_COS_C[n]);
  const double sn = swp ? C : S, cs = swp ? S : C;
  switch (k & 3) {
    case 0: c = cs; s = sn; break;
    case 1: c = -sn; s = cs; break;
    case 2: c = -cs; s = -sn; break;
    default: c = sn; s = -cs; break;
  }
}

// isotropic direction with mu on the x axis (C.4)
__device__ __forceinline__ void isotropic_dir(double a, double b, double &ux, double &uy, double &uz)
{
  const double mu = 2.0 * a - 1.0;
  double c, s;
  mc_sincos2pi(b, c, s);
  const double q = sqrt(fma(-mu, mu, 1.0));
  ux = mu; uy = q * c; uz = q * s;
}

// ------------------------------------------------------------ particle state
// 80-byte SoA record in five 16-byte chunks (north_star item 1)
// The four 16-byte chunks of position, time, direction and weight of one particle share one 64-byte line
// ("body"), the (id, packed state) chunks are an array of their own: the census close sorts on the ids alone
// and then gathers records in sorted order, and a random 64-byte line costs one DRAM access where four
// separate 16-byte gathers cost four (ncu: profiles/census_close_r2.md).  Streaming passes (source, pool entry
// and exit, comb output) touch every byte of a line either way.
struct Chunk {
  double2 *base;             // chunk c of record i at base[4 i]
  __device__ __forceinline__ double2 &operator[](size_t i) const { return base[4 * i]; }
  __device__ __forceinline__ double2 *operator+(size_t i) const { return base + 4 * i; }
};
struct Bank {
  Chunk xy, zt, uxy, uzw;
  ulonglong2 *idp;           // (pid, packed)
};

// packed: [63:40] ectr | [39:32] g | [31:22] ix | [21:12] iy | [11:2] iz | [1] inside | [0] spare
__device__ __forceinline__ uint64_t pack_state(uint32_t ectr, int g, int ix, int iy, int iz, int inside)
{
  return ((uint64_t)ectr << 40) | ((uint64_t)(uint32_t)g << 32) | ((uint64_t)(uint32_t)ix << 22) |
         ((uint64_t)(uint32_t)iy << 12) | ((uint64_t)(uint32_t)iz << 2) | ((uint64_t)(inside & 1) << 1);
}
__device__ __forceinline__ uint32_t pk_ectr(uint64_t p) { return (uint32_t)(p >> 40); }
__device__ __forceinline__ int pk_g(uint64_t p) { return (int)((p >> 32) & 0xFF); }
__device__ __forceinline__ int pk_ix(uint64_t p) { return (int)((p >> 22) & 0x3FF); }
__device__ __forceinline__ int pk_iy(uint64_t p) { return (int)((p >> 12) & 0x3FF); }
__device__ __forceinline__ int pk_iz(uint64_t p) { return (int)((p >> 2) & 0x3FF); }
__device__ __forceinline__ int pk_inside(uint64_t p) { return (int)((p >> 1) & 1); }

// ----------------------------------------------------------- problem tables
struct AxisHint { double p0, inv_w; };   // uniform finite plane table: origin and 1/width, else inv_w = 0
struct DevProblem {
  int n_mat, G;
  // per (m,g): sigma_t, sigma_s_row, sigma_f, nu  -> xs4[(m*G+g)*4 + k]
  const double *xs4;
  const double *cdf_s;     // [M][G][G]
  const double *cdf_chi;   // [M][G]
  const double *cdf_src;   // [G]
  const double *speed;     // [G]
  int nx, ny, nz;
  const double *px, *py, *pz;       // lattice planes
  const int8_t *mat_outer, *mat_inner; // [nz][ny][nx] (n_mat <= 127)
  const double *radius;
  int has_pins;
  int bc[6];
  int src_kind, src_isotropic;
  double src_lo[3], src_hi[3], src_dir[3], src_t0;
  double src_t1;                    // source with a time extent (C.17): birth time uniform in [src_t0, src_t1]; <= src_t0: pulse
  long long n_pins; const int *pin_cell;
  int tnx, tny, tnz, tnt;
  const double *tx, *ty, *tz, *tt;  // tally planes
  AxisHint hx, hy, hz, ht;          // uniform-table hints of the tally planes
  int aggregate_tally;              // warp-aggregate same-bin lanes before the RED (small hot tallies)
  int simple_tally;                 // tally plane tables bitwise equal to the lattice plane tables
  int planes_finite;                // every lattice plane is finite (nearest_plane in mcdc_pool.cu)
  long long tcross_off;             // offset of the time-crossing block in the tally (-1: off), include/mcdc.h
  // delayed neutrons (C.16): J precursor groups (0: all prompt); prompt yield [M][G], delayed yields
  // [M][G][J], decay constants [M][J], CDFs of the delayed spectra [M][J][G] (global memory: read at births only)
  int dn_J;
  const double *dn_nup, *dn_nu, *dn_lambda, *dn_cdf;
  double ic_w_roulette, ic_w_survive; // implicit capture (C.15): roulette below w_roulette (0: off) back to w_survive
  int march_min, march_iter_min, march_first;    // MARCH variants: see mcdc_pool.cu
  // quadric-surface CSG inside the one lattice cell (C.18) and moving surfaces (C.19); n_region = 0: lattice only
  int csg_n_surf, csg_n_region;
  const double *csg_coef;           // [n_surf][10]
  const int8_t *csg_rsurf;          // [n_region][8] signed surface id + 1, 0-terminated
  const int8_t *csg_rmat;           // [n_region]
  int mv_n_tau;
  const double *mv_tau, *mv_disp, *mv_vel;   // [n_tau], [n_surf][n_tau][3] displacement at / velocity after the break times
  double *tally;                    // current batch tally [tnt][G][tnz][tny][tnx] (+ the time-crossing block)
};

// direction-aware interval lookup (C.4): largest i with P[i] <= p, lower interval
// when exactly on a plane and moving down; clamped to [0, n-1].  Binary search.
__device__ __forceinline__ int find_interval(const double *__restrict__ P, int n, double p, double u)
{
  int lo = -1, hi = n + 1;       // invariant: P[lo] <= p (or lo = -1), P[hi] > p (or hi = n+1)
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(P + mid) <= p) lo = mid; else hi = mid;
  }
  if (lo >= 0 && __ldg(P + lo) == p && u < 0.0) lo -= 1;
  return min(max(lo, 0), n - 1);
}

// Same result as find_interval, reached from a guess: one probe of the guessed interval
// decides the strictly-inside and the exactly-on-a-plane cases (the on-plane rule is the
// definition's: largest i with P[i] <= p, minus one when moving down); anything else
// falls back to the search.  hint = (origin, 1/width) of a uniform finite table, else 0.
__device__ __forceinline__ int find_interval_fast(const double *__restrict__ P, int n, double p, double u,
                                                  const AxisHint h)
{
  int j = (h.inv_w > 0.0) ? (int)((p - h.p0) * h.inv_w) : 0;
  j = min(max(j, 0), n - 1);
  const double a = __ldg(P + j), b = __ldg(P + j + 1);
  if (a < p && p < b) return j;
  if (p == a) return max(u < 0.0 ? j - 1 : j, 0);
  if (p == b) return min(u < 0.0 ? j : j + 1, n - 1);
  return find_interval(P, n, p, u);
}

// the same two functions on plane tables that may live in shared memory (plain loads)
__device__ __forceinline__ int find_interval_any(const double *P, int n, double p, double u, const AxisHint h)
{
  int j = (h.inv_w > 0.0) ? (int)((p - h.p0) * h.inv_w) : 0;
  j = min(max(j, 0), n - 1);
  const double a = P[j], b = P[j + 1];
  if (a < p && p < b) return j;
  if (p == a) return max(u < 0.0 ? j - 1 : j, 0);
  if (p == b) return min(u < 0.0 ? j : j + 1, n - 1);
  int lo = -1, hi = n + 1;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (P[mid] <= p) lo = mid; else hi = mid;
  }
  if (lo >= 0 && P[lo] == p && u < 0.0) lo -= 1;
  return min(max(lo, 0), n - 1);
}
__device__ __forceinline__ double plane_dist_any(const double *P, int i, double p, double u)
{
  if (u == 0.0) return __longlong_as_double(0x7FF0000000000000ll);
  const double d = (P[i + (u > 0.0 ? 1 : 0)] - p) / u;
  return d < 0.0 ? 0.0 : d;
}

// distance along u to the next plane of interval i, clamped at 0 (C.5 step 4, App. C)
__device__ __forceinline__ double plane_dist(const double *__restrict__ P, int i, double p, double u)
{
  if (u == 0.0) return __longlong_as_double(0x7FF0000000000000ll);
  const double edge = __ldg(P + i + (u > 0.0 ? 1 : 0));
  const double d = (edge - p) / u;
  return d < 0.0 ? 0.0 : d;
}

// z-cylinder distance with the logical region flag selecting the root (App. C.1)
__device__ __forceinline__ double cyl_dist(double x, double y, double ux, double uy, double cx,
                                           double cy, double R, int inside)
{
  const double INF = __longlong_as_double(0x7FF0000000000000ll);
  const double dx = x - cx, dy = y - cy;
  const double A = fma(ux, ux, uy * uy);
  if (A == 0.0) return INF;
  const double Bh = fma(dx, ux, dy * uy);
  const double Cc = fma(dx, dx, dy * dy) - R * R;
  double D = fma(Bh, Bh, -(A * Cc));
  double s;
  if (inside) {
    if (D <= 0.0) D = 0.0;
    s = (Bh <= 0.0) ? (sqrt(D) - Bh) / A : -Cc / (sqrt(D) + Bh);
  } else {
    if (Bh >= 0.0 || D <= 0.0) return INF;
    s = Cc / (sqrt(D) - Bh);
  }
  return s < 0.0 ? 0.0 : s;
}

// ------------------------------------------------ quadric-surface CSG (C.18), moving surfaces (C.19)
// Plain IEEE expressions evaluated left to right as written (compiled with -fmad=false): the definition's.
constexpr int CSG_NO_REGION = 1023;      // value of the ix field of a particle that is in no region (lost at its next flight)

__device__ __forceinline__ double quad_eval(const double *q, double x, double y, double z)
{
  return q[0] * x * x + q[1] * y * y + q[2] * z * z + q[3] * x * y + q[4] * y * z + q[5] * z * x +
         q[6] * x + q[7] * y + q[8] * z + q[9];
}

// first s >= 0 at which sense * f(r + s u) turns negative (the particle is logically where it is positive)
__device__ __forceinline__ double quadric_dist(const double *q, double sense, double x, double y, double z,
                                               double ux, double uy, double uz)
{
  const double INF = __longlong_as_double(0x7FF0000000000000ll);
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

// displacement of surface s at time t and its velocity there
__device__ __forceinline__ void surf_motion(const DevProblem &P, int s, double t, double d[3], double vel[3])
{
  d[0] = d[1] = d[2] = 0.0; vel[0] = vel[1] = vel[2] = 0.0;
  const int n = P.mv_n_tau;
  if (n == 0) return;
  int k = -1;
  for (int j = 0; j < n; ++j) if (__ldg(P.mv_tau + j) <= t) k = j;
  const double *D = P.mv_disp + (size_t)s * n * 3, *V = P.mv_vel + (size_t)s * n * 3;
  if (k < 0) { d[0] = __ldg(D); d[1] = __ldg(D + 1); d[2] = __ldg(D + 2); return; }
  const double dt = t - __ldg(P.mv_tau + k);
#pragma unroll
  for (int i = 0; i < 3; ++i) { vel[i] = __ldg(V + k * 3 + i); d[i] = __ldg(D + k * 3 + i) + vel[i] * dt; }
}

__device__ __forceinline__ int surf_side(const DevProblem &P, const double *coef, int s, double x, double y, double z, double t)
{
  double d[3], vel[3];
  surf_motion(P, s, t, d, vel);
  return quad_eval(coef + s * 10, x - d[0], y - d[1], z - d[2]) > 0.0 ? 1 : -1;
}

// region that holds the point: all sides from the coordinates (from < 0), or after the particle of region `from`
// crossed surface `crossed`: the logical sides of `from` with that one flipped, coordinates only for surfaces
// `from` does not know.  First match in index order; -1: none.
__device__ __forceinline__ int find_region(const DevProblem &P, const double *coef, int from, int crossed,
                                           double x, double y, double z, double t)
{
  for (int q = 0; q < P.csg_n_region; ++q) {
    bool ok = true;
    for (int j = 0; j < 8 && ok; ++j) {
      const int e = (int)__ldg(P.csg_rsurf + q * 8 + j);
      if (e == 0) break;
      const int sf = (e > 0 ? e : -e) - 1, want = e > 0 ? 1 : -1;
      int have = 0;
      if (from >= 0)
        for (int i = 0; i < 8; ++i) {
          const int f = (int)__ldg(P.csg_rsurf + from * 8 + i);
          if (f == 0) break;
          if ((f > 0 ? f : -f) - 1 == sf) { have = f > 0 ? 1 : -1; if (sf == crossed) have = -have; break; }
        }
      if (have == 0) have = surf_side(P, coef, sf, x, y, z, t);
      if (have != want) ok = false;
    }
    if (ok) return q;
  }
  return -1;
}

}  // namespace mcdc
