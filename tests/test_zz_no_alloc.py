"""mcdc_batch_stats_noalloc (include/mcdc.h): the entry point that allocates no device memory — batch
close-out + mean / standard error with the running sums in a fixed device array of the library — against the
workspace path (mcdc_run over the same batches + mcdc_tally_read), on two calls in a row that share the array.
Collected last (file name): a failure here hides no other test under pytest -x."""
import numpy as np
import pytest

import mcdc_inputs as mi
from parity import RTOL

pytestmark = pytest.mark.gpu


def _existing_path(make_cfg, n_batch, monkeypatch):
    """Workspace path: one run of n_batch batches -> mean, standard error; and the raw tally of every batch from
    one-batch runs with seed + b (include/mcdc.h: batch b uses Philox stream seed + b), on the device."""
    import torch
    from paper_2305_07636_b200 import Problem
    monkeypatch.setenv("MCDC_PIPELINES", "1")          # batches fold into the sums in order 0, 1, 2, ...
    cfg = make_cfg(n_batch)
    p = Problem(cfg).run()
    mean, err = p.tally(0).ravel().copy(), p.tally(1).ravel().copy()
    p.close()
    rows = []
    for b in range(n_batch):
        c1 = make_cfg(1)
        c1["run"]["seed"] = cfg["run"]["seed"] + b
        q = Problem(c1).run()
        rows.append(q.tally_device(2).reshape(-1).clone())
        q.close()
    return torch.stack(rows).contiguous(), cfg["run"]["n_hist_per_batch"], mean, err


def _check(got_mean, got_err, mean, err, what):
    zero = mean == 0.0
    assert np.all(got_mean[zero] == 0.0), what
    rel = np.abs(got_mean - mean) / np.maximum(np.abs(mean), 1e-300)
    assert np.all(rel[~zero] <= RTOL), f"{what}: mean, max rel err {rel[~zero].max():.3e}"
    # the rule of tests/parity.py for the standard error (sqrt of a difference of sums)
    assert np.all(np.abs(got_err * got_err - err * err) <= 4 * RTOL * mean * mean + 1e-300), f"{what}: standard error"


def test_no_alloc_batch_stats_match_the_workspace_path_twice_in_a_row(monkeypatch):
    import torch
    from paper_2305_07636_b200 import batch_stats_noalloc
    a = _existing_path(lambda nb: mi.config2(n_hist=20_000, n_batch=nb, seed=5), 3, monkeypatch)       # 100 x 200 bins
    b = _existing_path(lambda nb: mi.config4(n_hist=4_000, n_batch=nb, seed=9, t_end=2e-6), 4, monkeypatch)
    assert a[0].shape[1] != b[0].shape[1] and np.count_nonzero(a[2]) > 1000 and np.count_nonzero(b[2]) > 1000
    outs = []
    for rows, n_hist, _, _ in (a, b, a):               # back to back on one stream: the calls share the scratch array
        mean = torch.full((rows.shape[1],), float("nan"), dtype=torch.float64, device="cuda")
        err = torch.full_like(mean, float("nan"))
        batch_stats_noalloc(rows, n_hist, mean, err)
        outs.append((mean, err))
    torch.cuda.synchronize()
    for (mean, err), ref, what in zip(outs, (a, b, a), ("first call", "second call", "third call")):
        _check(mean.cpu().numpy(), err.cpu().numpy(), ref[2], ref[3], what)
    # same kernels, same order of operations: the first and the third call agree bit for bit
    assert torch.equal(outs[0][0], outs[2][0]) and torch.equal(outs[0][1], outs[2][1])
    # mean only, one batch: no standard error asked for
    mean = torch.empty(a[0].shape[1], dtype=torch.float64, device="cuda")
    batch_stats_noalloc(a[0][:1].contiguous(), a[1], mean)
    torch.cuda.synchronize()
    assert torch.equal(mean, a[0][0] / torch.full_like(mean, float(a[1])))    # (a tensor divisor: IEEE division per element)


def test_no_alloc_rejects_sizes_beyond_the_fixed_array():
    import torch
    from paper_2305_07636_b200 import batch_stats_noalloc, McdcError, NOALLOC_MAX_BINS
    n = NOALLOC_MAX_BINS + 1
    rows = torch.zeros((1, n), dtype=torch.float64, device="cuda")
    mean = torch.zeros(n, dtype=torch.float64, device="cuda")
    with pytest.raises(McdcError, match="MCDC_NOALLOC_MAX_BINS"):
        batch_stats_noalloc(rows, 1.0, mean)
    # the largest size the array holds still runs
    n = NOALLOC_MAX_BINS
    rows = torch.rand((2, n), dtype=torch.float64, device="cuda")
    mean, err = torch.empty(n, dtype=torch.float64, device="cuda"), torch.empty(n, dtype=torch.float64, device="cuda")
    batch_stats_noalloc(rows, 2.0, mean, err)
    torch.cuda.synchronize()
    assert torch.allclose(mean, rows.sum(0) / 4.0, rtol=1e-14, atol=0)
    assert torch.allclose(err, (rows[0] - rows[1]).abs() / 4.0, rtol=1e-6, atol=1e-7)   # (cancellation in sum x^2 / B - mean^2 where the two rows nearly agree)
