"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  Walkers shard across ranks with no
data-path collective; timing is the max over ranks, accepted moves are summed."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1708_00744_b200 import dist as qdist
from paper_1708_00744_b200 import inputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    batch, N = 3, 16
    wl = inputs.make_workload(batch, N, 8, seed=qdist.rank_seed(1, rank, batch))
    accepted = int(wl.bernoulli_mask(0.5).sum())
    ms = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms_max, acc_sum = qdist.combine(ms, accepted)
    out[rank] = (ms_max, acc_sum, accepted, float(wl.A[0, 0, 0]))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo_max_time_sum_accepted_disjoint_walkers():
    world = 2
    with mp.Manager() as man:
        out = man.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        r0, r1 = out[0], out[1]
    assert r0[0] == r1[0] == 15.0                        # max over ranks
    assert r0[1] == r1[1] == r0[2] + r1[2]               # sum of accepted moves
    assert r0[3] != r1[3]                                # different walkers on the two ranks
    # rank 0 reproduces the single-GPU workload, rank 1 continues the walker seeds
    a = inputs.make_workload(6, 16, 8, seed=1)
    b = inputs.make_workload(3, 16, 8, seed=qdist.rank_seed(1, 1, 3))
    assert np.array_equal(a.A[3:], b.A) and np.array_equal(a.proposals[:, 3:], b.proposals)
    assert qdist.moves_per_second(30.0, 2, 600) == 600 / 15e-3


def test_combine_without_process_group_is_identity():
    assert qdist.combine(3.5, 7) == (3.5, 7)
    assert qdist.rank_seed(1, 0, 16) == 1
