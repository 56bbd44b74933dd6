"""Host-side logic of the multi-GPU (batch replica) path, world_size 2 and 3 over gloo on CPU.
The per-batch engine here is the oracle (tests may use it); on GPUs it is Problem.run followed by
replicas.combine (tests/test_gpu_parity.py::test_replica_combine_*)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

N_HIST, SEED = 2000, 3


def _cfg():
    import mcdc_inputs as mi
    return mi.config2(n_hist=N_HIST, n_batch=1)


def _worker(rank, world, port, n_batch, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import Oracle, COUNTER_NAMES
    from paper_2305_07636_b200 import replicas
    o = Oracle(_cfg())

    def run_batch(seed_b):
        o.run(seed=seed_b, n_hist_per_batch=N_HIST, n_batch=1)
        return o.tally(2), o.counters(0)

    s1, s2, c = replicas.run_replicated(run_batch, n_batch, SEED, o.shape, rank, world)
    s1, s2, c = replicas.all_reduce_replicas(s1, s2, c, COUNTER_NAMES)
    if rank == 0:
        torch.save(dict(s1=s1, s2=s2, counters=c), out)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,n_batch", [(2, 5), (3, 2)])     # (3, 2): a rank without a batch still joins the collectives
def test_ranks_equal_one_process(tmp_path, world, n_batch):
    from paper_2305_07636_b200 import replicas
    assert replicas.my_batches(5, 0, 2) == [0, 2, 4] and replicas.my_batches(5, 1, 2) == [1, 3]
    assert replicas.my_batches(2, 2, 3) == []
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(world, 29500 + (os.getpid() + 7 * world) % 2000, n_batch, out), nprocs=world, join=True)
    got = torch.load(out)
    from oracle import Oracle, COUNTER_NAMES
    ref = Oracle(_cfg())
    s1 = np.zeros(ref.shape); s2 = np.zeros(ref.shape)
    tot = {n: 0 for n in COUNTER_NAMES}
    for b in range(n_batch):
        ref.run(seed=SEED + b, n_hist_per_batch=N_HIST, n_batch=1)
        x = ref.tally(2)
        s1 += x; s2 += x * x
        for n, v in ref.counters(0).items():
            tot[n] = (tot[n] + v) % (1 << 64)
    np.testing.assert_allclose(got["s1"].numpy(), s1, rtol=1e-13, atol=0)
    np.testing.assert_allclose(got["s2"].numpy(), s2, rtol=1e-13, atol=0)
    assert got["counters"] == tot
    # and the sums are what the oracle's own multi-batch statistics are made of
    ref.run(seed=SEED, n_hist_per_batch=N_HIST, n_batch=n_batch)
    np.testing.assert_allclose(s1 / (n_batch * N_HIST), ref.tally(0), rtol=1e-12, atol=0)
