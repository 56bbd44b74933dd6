// mcdc_kernels.cuh — shared declarations of the event kernels and the host driver.
#pragma once
#include "mcdc_device.cuh"

namespace mcdc {

constexpr int BS = 256;           // threads per block of every event kernel
constexpr int NWARP = BS / 32;
constexpr int N_CNT = 16;

// counter slots (same order as mcdc_counters in include/mcdc.h)
enum { K_SOURCE, K_FLIGHTS, K_SEGMENTS, K_COLLISIONS, K_SCATTERS, K_CAPTURES, K_FISSIONS,
       K_SECONDARIES, K_CROSSINGS, K_REFLECTIONS, K_LEAKS, K_CENSUS, K_COMB_IN, K_COMB_OUT,
       K_LOST, K_FINGERPRINT };
// terminal events entering the fingerprint
enum { END_CAPTURE = 0, END_FISSION = 1, END_LEAK = 2, END_CENSUS = 3, END_LOST = 4 };

// Device-resident control block: queue lengths and the parameters of the current
// census step, so the same launches can be replayed without host-side arguments.
struct Ctl {
  uint32_t n_active, n_next, n_coll, n_census;
  uint32_t bank_tail, parity, overflow, iter;
  uint32_t wq_head, wq_tail, wq_pending, fetch;    // fetch: next unreserved entry of the active queue (REFILL)   // device-side work queue of the tail kernel
  double t_k;
  unsigned long long seedb;
  uint32_t last_step, step_k1;
  uint32_t comb_front, comb_back;  // comb: survivors with long histories ahead are written from the front of the bank, the rest from the back
  uint32_t spill_lo, spill_limit;  // pool kernel: window of the active bank that takes children the pools cannot hold
  unsigned long long *cnt;       // counter row of the current (batch, step)
  double eig_k;                  // k-eigenvalue mode (C.14): k the running generation divides its fission yield by
  uint32_t score;                // ... and whether the generation scores the tally (active cycle)
  uint32_t pool_chunk;           // pool kernel: entries of the active bank a warp reserves per atomic (32 | 128)
  uint32_t spill_seen;           // pool kernel: a launch left spilled children behind and the host did not wait for it
  uint32_t err_code, err_step;   // first error the device found in this batch (E_* below), and its step
};
enum { E_NONE = 0, E_EIG_YIELD = 1 /* nu / k > 7 */, E_EIG_DIED = 2 /* a generation without children */ };

struct Queues {
  uint32_t *q[2];                // active / next, selected by Ctl::parity
  uint32_t *coll;                // collision queue
  uint32_t *census;              // census list of the current step
  uint32_t capacity;             // bank slots = max entries of any queue
};

struct TableLayout {             // offsets (in doubles) into the staged table block
  int xs4, cdf_s, cdf_chi, cdf_src, speed, total;
};

}  // namespace mcdc
