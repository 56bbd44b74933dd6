"""Writes mcdc_inputs/config5_scale.json: the nu*Sigma_f multiplier that makes config 5
'slightly supercritical' (BASELINE.json:11; reading S17).

Bisection on the scalar so that the pre-comb population ratio N_k / M, averaged over
census steps 10..19 of a 1e5-history pilot, lies in [1.00, 1.02] (target 1.01).
Calls only oracle/ (the CUDA path is never used to produce stored values).

    python -m mcdc_inputs.calibrate_config5
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import mcdc_inputs as mi  # noqa: E402
from oracle import Oracle  # noqa: E402

N = 100_000


def ratio(scale):
    o = Oracle(mi.config5(n_hist=N, n_batch=1, nusf_scale=scale)).run()
    r = np.array([o.counters(0, k)["comb_in"] / N for k in range(9, 19)])
    o.close()
    return float(r.mean())


def main():
    lo, hi = 1.0, 8.0
    rl, rh = ratio(lo), ratio(hi)
    print("bracket", lo, rl, hi, rh, flush=True)
    assert rl < 1.01 < rh
    for _ in range(12):
        mid = 0.5 * (lo + hi)
        r = ratio(mid)
        print(mid, r, flush=True)
        if 1.005 <= r <= 1.015:
            lo = hi = mid
            break
        if r < 1.01:
            lo = mid
        else:
            hi = mid
    scale = 0.5 * (lo + hi)
    out = dict(nusf_scale=scale, pilot_ratio=ratio(scale), pilot_histories=N,
               rule="mean over census steps 10..19 of N_k/M in [1.00,1.02]")
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config5_scale.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(out)


if __name__ == "__main__":
    main()
