"""Batch-replica sharding across ranks.

Histories are independent and every batch b uses the Philox stream seed + b, so the path
shards by batch with no exchange step: rank r runs batches r, r + W, r + 2W, ... on its own
GPU and the per-batch raw tallies are folded into sum x / sum x^2; ONE all-reduce at the end
combines the replicas (NCCL over NVLink on GPUs, gloo in the CPU tests).  Counters are
integer sums and combine the same way.
"""
import torch
import torch.distributed as dist


def my_batches(n_batch_total, rank, world):
    """Batch indices owned by `rank` (round-robin, so every rank gets floor or ceil of B/W)."""
    return list(range(rank, n_batch_total, world))


def run_replicated(run_batch, n_batch_total, seed, rank=0, world=1, device="cpu"):
    """run_batch(seed_b) -> (raw tally tensor/array of one batch, dict of integer counters).

    Returns (mean per source particle not yet divided by N: sum1, sum2, counters) after the
    all-reduce; every rank holds the full result."""
    s1 = s2 = None
    counters = {}
    for b in my_batches(n_batch_total, rank, world):
        x, c = run_batch(seed + b)
        x = torch.as_tensor(x, dtype=torch.float64, device=device)
        if s1 is None:
            s1, s2 = torch.zeros_like(x), torch.zeros_like(x)
        s1 += x
        s2 += x * x
        for k, v in c.items():
            counters[k] = counters.get(k, 0) + int(v)
    return s1, s2, counters


def all_reduce_replicas(s1, s2, counters, names):
    """Sum the replicas' sums and counters over the default process group (no-op if W = 1).
    Counters travel as int64 (wrapping sums such as the fingerprint stay exact modulo 2^64)."""
    c = torch.tensor([(counters.get(n, 0) + (1 << 63)) % (1 << 64) - (1 << 63) for n in names],
                     dtype=torch.int64, device=s1.device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(s1, op=dist.ReduceOp.SUM)
        dist.all_reduce(s2, op=dist.ReduceOp.SUM)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    out = {n: int(v) % (1 << 64) for n, v in zip(names, c.tolist())}
    return s1, s2, out


def statistics(s1, s2, n_batch_total, n_hist_per_batch):
    """Mean per source particle and its standard error over batches (same formulas as the library)."""
    B, N = float(n_batch_total), float(n_hist_per_batch)
    mean = s1 / (B * N)
    if n_batch_total < 2:
        return mean, torch.zeros_like(mean)
    m = s1 / B
    var = torch.clamp((s2 / B - m * m) * (B / (B - 1.0)), min=0.0)
    return mean, torch.sqrt(var / B) / N
