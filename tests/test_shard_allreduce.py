"""The N > 1 path of the sharded build on CPU (world_size 2, gloo).  The kernels deal their work round-robin over the
ranks (pbc_jk_set_shard; the sum of the ranks' partial J and K is the full matrix -- checked on the GPU by
tests/test_parity_gpu.py::test_shards_sum_to_full_build); what runs on the host is the ONE collective of the path, the
all-reduce of [J; K] (binding.allreduce_jk).  Here two gloo ranks hold complementary partial matrices and must both
end with the sums, on the one-message path (J and K back to back) and on the staged path."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2410_22278_b200.binding import allreduce_jk
    n = 37
    rng = np.random.default_rng(123)
    Jfull, Kfull = rng.standard_normal((n, n)), rng.standard_normal((n, n))
    mask = (np.arange(n * n).reshape(n, n) % world) == rank        # this rank's share of every matrix
    ok = True
    # (a) J and K as the two halves of one buffer: one message
    JK = torch.zeros((2, n, n), dtype=torch.float64)
    JK[0] = torch.from_numpy(Jfull * mask)
    JK[1] = torch.from_numpy(Kfull * mask)
    allreduce_jk(JK[0], JK[1])
    ok &= np.allclose(JK[0].numpy(), Jfull, atol=0, rtol=0) and np.allclose(JK[1].numpy(), Kfull, atol=0, rtol=0)
    # (b) separate tensors: staged through one concatenated buffer
    J = torch.from_numpy(Jfull * mask).clone()
    K = torch.from_numpy(Kfull * mask).clone()
    allreduce_jk(J, K)
    ok &= np.array_equal(J.numpy(), Jfull) and np.array_equal(K.numpy(), Kfull)
    # (c) only one of the two matrices
    J = torch.from_numpy(Jfull * mask).clone()
    allreduce_jk(J, None)
    ok &= np.array_equal(J.numpy(), Jfull)
    out[rank] = bool(ok)
    dist.destroy_process_group()


def test_allreduce_jk_two_ranks_gloo():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29741, out), nprocs=world, join=True)
        assert dict(out) == {0: True, 1: True}


def test_allreduce_jk_is_a_no_op_without_a_process_group():
    sys.path.insert(0, ROOT)
    from paper_2410_22278_b200.binding import allreduce_jk
    J = torch.ones((3, 3), dtype=torch.float64)
    allreduce_jk(J, None)
    assert float(J.sum()) == 9.0
