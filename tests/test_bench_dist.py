"""The multi-rank bookkeeping of bench.py on CPU (gloo, world size 2): the path has no inter-GPU step
("replicas only"), so all that N > 1 adds is max-over-ranks timing and the whole-job sum."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    sec = bench.max_over_ranks(1.0 + rank, dist, "cpu")          # rank 1 is the slow one
    value = bench.whole_job_value(1000, 4, world, sec)
    dist.barrier()
    out[rank] = (sec, value)
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29541, out), nprocs=world, join=True)
    for rank in range(world):
        sec, value = out[rank]
        assert sec == 2.0                                           # the max, on every rank
        assert value == 2 * 1000 * 4 / 2.0                          # all ranks' work over the slowest time


def test_dof_update_count_follows_the_levels():
    import numpy as np
    import bench
    # 3 levels: K_l * 2^level * 4 Np
    levels = np.array([0] * 10 + [1] * 5 + [2] * 2)
    assert bench.dof_updates_per_global_step(levels, 20) == (10 * 1 + 5 * 2 + 2 * 4) * 4 * 20
