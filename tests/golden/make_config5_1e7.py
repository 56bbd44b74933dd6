"""Writes tests/golden/config5_1e7_seed0.npz: what the ORACLE computes for one full batch of
BASELINE.json config 5 at the batch size bench.py times (1e7 histories, seed 0, 20 census steps
with comb to 1e7).  Calls only oracle/ and mcdc_inputs/ (array builders):
no stored value ever comes from the CUDA path.

Stored (the raw batch tally has 36.7e6 bins = 294 MB, too large to commit):
  counters   [20][16] uint64   every counter row of the batch, fingerprints included
  plane_sums [20][7]  float64  sum over the 64^3 spatial bins of every (time bin, group) plane
                               (math.fsum: exactly rounded, so independent of summation order)
  nonzero    [20][7]  int64    number of non-zero bins per plane
  idx        [N_SAMPLE] int64  flat indices of seeded-random bins (numpy default_rng(5))
  val        [N_SAMPLE] float64 their raw values (which = 2)
  zero_idx   [<= N_ZERO] int64 flat indices of seeded-random bins that are exactly 0.0

    python tests/golden/make_config5_1e7.py        (about 15 minutes, one core, ~6 GB)
"""
import math
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import mcdc_inputs as mi  # noqa: E402
from oracle import Oracle, COUNTER_NAMES  # noqa: E402

N_HIST = 10_000_000
N_SAMPLE = 100_000
N_ZERO = 20_000
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config5_1e7_seed0.npz")


def main(n_hist=N_HIST, out=OUT):
    cfg = mi.config5(n_hist=n_hist, n_batch=1, seed=0)
    t0 = time.perf_counter()
    o = Oracle(cfg).run()
    dt = time.perf_counter() - t0
    counters = np.array([[o.counters(0, k)[n] for n in COUNTER_NAMES] for k in range(o.n_steps)], dtype=np.uint64)
    raw = o.tally(2)
    nt, G = raw.shape[:2]
    plane_sums = np.array([[math.fsum(raw[t, g].ravel()) for g in range(G)] for t in range(nt)])
    nonzero = np.array([[int(np.count_nonzero(raw[t, g])) for g in range(G)] for t in range(nt)], dtype=np.int64)
    flat = raw.ravel()
    rng = np.random.default_rng(5)
    idx = np.sort(rng.choice(flat.size, N_SAMPLE, replace=False)).astype(np.int64)
    zeros = np.flatnonzero(flat == 0.0)
    zero_idx = np.sort(rng.choice(zeros, min(N_ZERO, zeros.size), replace=False)).astype(np.int64) if zeros.size else zeros
    np.savez_compressed(out, counters=counters, plane_sums=plane_sums, nonzero=nonzero, idx=idx, val=flat[idx],
                        zero_idx=zero_idx, n_hist=np.int64(n_hist), oracle_seconds=np.float64(dt))
    print(f"wrote {out}: {n_hist} histories in {dt:.0f} s, {int(counters[:, 1].sum())} flights, "
          f"{int(np.count_nonzero(flat))} non-zero bins, {zeros.size} zero bins")


if __name__ == "__main__":
    if len(sys.argv) > 2:
        main(int(sys.argv[1]), sys.argv[2])
    else:
        main()
