"""Host logic of bench.py on CPU: the roofline numerator and the N > 1 aggregation (max over ranks through
torch.distributed; gloo here, nccl on the GPU box)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def test_alg_flops_formula():
    st = {"alg_sum_n2": 1000, "alg_sum_n": 100, "alg_incidence": 10}
    # unique orbital pairs n(n+1) + V dV scaling n + 120 per (point, atom)
    assert bench.alg_flops(st) == 1000 + 100 + 100 + 120 * 10


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = bench.max_over_ranks([0.1 * (rank + 1), 1.0 - 0.25 * rank], torch.device("cpu"), world)
    out[rank] = t
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, 29613, out), nprocs=world, join=True)
        for r in range(world):
            assert np.allclose(out[r], [0.2, 1.0])
    # whole-job value for replicas: N * points / slowest rank
    assert bench.job_value(1000, 0.2, world) == 2 * 1000 / 0.2
