"""N > 1 path of bench.py ("replicas only") on CPU: two gloo ranks, no GPU.  Checks the seeded
per-rank initial states and the only collective of the job (max of the times, sum of the work)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402
from ocp_inputs import make_config  # noqa: E402


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = make_config("C1")
    x0 = bench.replica_x0(cfg, rank)
    # rank r took (10 + r) ms on the device, (20 - r) ms end to end, 5 + r iterations, 6 + r factorizations, 3 steps, 40 launches
    res = bench.aggregate_over_ranks(dist, world, torch.device("cpu"), 10.0 + rank, 20.0 - rank, 5 + rank, 6 + rank, 3, 40)
    out[rank] = (x0, res)
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_aggregate_and_seed():
    world = 2
    port = 29500 + (os.getpid() % 2000)
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        (x0a, ra), (x0b, rb) = out[0], out[1]
    assert ra == rb == (11.0, 20.0, 11, 13, 6, 80)           # max times, summed work
    cfg = make_config("C1")
    assert np.array_equal(x0a, np.asarray(cfg.x0, dtype=np.float64))          # rank 0 = the config's own x0
    assert not np.array_equal(x0a, x0b) and x0b.shape == x0a.shape            # rank 1 = a seeded perturbation of it
    assert np.all(x0b >= cfg.x0_clip[0]) and np.all(x0b <= cfg.x0_clip[1])
    assert np.array_equal(x0b, bench.replica_x0(cfg, 1))                      # deterministic


def test_single_rank_is_identity():
    assert bench.aggregate_over_ranks(None, 1, None, 1.5, 2.5, 7, 8, 2, 30) == (1.5, 2.5, 7, 8, 2, 30)
