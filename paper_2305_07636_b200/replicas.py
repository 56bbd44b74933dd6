"""Batch-replica sharding across ranks.

Histories are independent and every batch b uses the Philox stream seed + b, so the path shards by
batch with no exchange step: rank r runs batches r, r + W, r + 2W, ... on its own GPU and folds them
into its running sums sum x / sum x^2; ONE sum all-reduce at the end combines the replicas (NCCL over
NVLink on GPUs, in place on the library's workspace; gloo in the CPU tests).  Counters are wrapping
integer sums and combine the same way.  No statistics are computed here: after `combine`, the library's
own mcdc_tally_read returns the mean and standard error over all ranks' batches.
"""
import torch
import torch.distributed as dist


def my_batches(n_batch_total, rank, world):
    """Batch indices owned by `rank` (round-robin, so every rank gets floor or ceil of B/W)."""
    return list(range(rank, n_batch_total, world))


def _world():
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def combine(problem, group=None):
    """All-reduce the running sums and the counters of `problem` (a binding.Problem after run()) over
    the process group, in place on its device workspace, then tell the library how many replicas were
    summed.  Every rank must have run the same number of batches of the same size."""
    world = _world()
    if world > 1:
        sums, cnt = problem.replica_views()
        dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(cnt, op=dist.ReduceOp.SUM, group=group)    # int64 wraps like uint64: exact
        torch.cuda.current_stream().synchronize()
    problem.replica_commit(world)
    return problem


def run_replicated(run_batch, n_batch_total, seed, shape, rank=0, world=1, device="cpu"):
    """Host-side form of the same scheme for engines that return one batch at a time:
    run_batch(seed_b) -> (raw tally of one batch, dict of integer counters).  Returns this rank's
    (sum x, sum x^2, counters); a rank that owns no batch (world > n_batch_total) returns zeros of
    `shape`, so that it can still take part in the collectives."""
    s1 = torch.zeros(shape, dtype=torch.float64, device=device)
    s2 = torch.zeros(shape, dtype=torch.float64, device=device)
    counters = {}
    for b in my_batches(n_batch_total, rank, world):
        x, c = run_batch(seed + b)
        x = torch.as_tensor(x, dtype=torch.float64, device=device).reshape(shape)
        s1 += x
        s2 += x * x
        for k, v in c.items():
            counters[k] = (counters.get(k, 0) + int(v)) % (1 << 64)
    return s1, s2, counters


def all_reduce_replicas(s1, s2, counters, names, group=None):
    """Sum the ranks' sums and counters over the process group (no-op if W = 1).  Counters travel as
    int64 (wrapping sums such as the fingerprint stay exact modulo 2^64)."""
    c = torch.tensor([(counters.get(n, 0) + (1 << 63)) % (1 << 64) - (1 << 63) for n in names],
                     dtype=torch.int64, device=s1.device)
    if _world() > 1:
        dist.all_reduce(s1, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(s2, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(c, op=dist.ReduceOp.SUM, group=group)
    out = {n: int(v) % (1 << 64) for n, v in zip(names, c.tolist())}
    return s1, s2, out
