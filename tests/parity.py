"""Shared comparison rule of the GPU-vs-oracle parity tests (DESIGN.md §3 C.12)."""
import numpy as np

RTOL = 1e-9   # north_star: "every fp64 tally bin within 1e-9 relative"


def compare(gpu, orc, n_batch, n_steps, what=""):
    """Counters equal as integers per (batch, step), fingerprint included; tallies within RTOL,
    bins that are exactly zero in the oracle exactly zero on the GPU."""
    for b in range(n_batch):
        for k in range(n_steps):
            cg, co = gpu.counters(b, k), orc.counters(b, k)
            assert cg == co, f"{what} batch {b} step {k}: " + str({n: (cg[n], co[n]) for n in cg if cg[n] != co[n]})
    for which in (2, 0, 1):
        a, r = gpu.tally(which), orc.tally(which)
        assert a.shape == r.shape
        zero = r == 0.0
        assert np.all(a[zero] == 0.0), f"{what} which={which}: {np.count_nonzero(a[zero])} bins not exactly zero"
        if which == 1:
            # the standard error is sqrt of a difference of sums (sum x^2 / B - mean^2): a 1e-9
            # relative difference of the sums shows up as 4e-9 * mean^2 in the variance
            mean = orc.tally(0)
            assert np.all(np.abs(a * a - r * r) <= 4 * RTOL * mean * mean + 1e-300), f"{what} which=1"
            continue
        err = np.abs(a - r) / np.maximum(np.maximum(np.abs(a), np.abs(r)), 1e-300)
        assert np.all(err[~zero] <= RTOL), f"{what} which={which}: max rel err {err[~zero].max():.3e}"
