"""Host-side logic of the multi-GPU (batch replica) path, world_size 2 over gloo on CPU.
The per-batch engine here is the oracle (tests may use it); on GPUs it is Problem.run."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

N_BATCH, N_HIST, SEED = 5, 2000, 3


def _cfg():
    import mcdc_inputs as mi
    return mi.config2(n_hist=N_HIST, n_batch=1)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import Oracle, COUNTER_NAMES
    from paper_2305_07636_b200 import replicas
    o = Oracle(_cfg())

    def run_batch(seed_b):
        o.run(seed=seed_b, n_hist_per_batch=N_HIST, n_batch=1)
        return o.tally(2), o.counters(0)

    s1, s2, c = replicas.run_replicated(run_batch, N_BATCH, SEED, rank, world)
    s1, s2, c = replicas.all_reduce_replicas(s1, s2, c, COUNTER_NAMES)
    mean, se = replicas.statistics(s1, s2, N_BATCH, N_HIST)
    if rank == 0:
        torch.save(dict(mean=mean, se=se, counters=c), out)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_equal_one_process(tmp_path):
    from paper_2305_07636_b200 import replicas
    assert replicas.my_batches(5, 0, 2) == [0, 2, 4] and replicas.my_batches(5, 1, 2) == [1, 3]
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, 29500 + os.getpid() % 2000, out), nprocs=2, join=True)
    got = torch.load(out)
    from oracle import Oracle, COUNTER_NAMES
    ref = Oracle(_cfg()).run(seed=SEED, n_hist_per_batch=N_HIST, n_batch=N_BATCH)
    np.testing.assert_allclose(got["mean"].numpy(), ref.tally(0), rtol=1e-12, atol=0)
    np.testing.assert_allclose(got["se"].numpy(), ref.tally(1), rtol=1e-6, atol=1e-18)
    tot = {n: 0 for n in COUNTER_NAMES}
    for b in range(N_BATCH):
        for n, v in ref.counters(b).items():
            tot[n] = (tot[n] + v) % (1 << 64)
    assert got["counters"] == tot
