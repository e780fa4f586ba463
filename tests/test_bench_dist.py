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


def _survey_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    nshots = 5
    mine = bench.shots_of_rank(nshots, rank, world)
    # stand-in for the per-rank stacked image: shot s contributes (s + 1) at entry s and 1 everywhere
    img = torch.zeros(8, dtype=torch.float64)
    for s in mine:
        img += 1.0
        img[s] += s + 1
    bench.stack_images(img, dist)
    out[rank] = (mine, img.tolist())
    dist.destroy_process_group()


def test_survey_shot_split_and_image_sum_gloo():
    """Shot-per-rank survey: every shot is done by exactly one rank and the one collective, the image
    all-reduce, gives every rank the sum over ALL shots."""
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_survey_worker, args=(world, 29543, out), nprocs=world, join=True)
    shots = sorted(out[0][0] + out[1][0])
    assert shots == [0, 1, 2, 3, 4] and not set(out[0][0]) & set(out[1][0])
    want = [5.0 + (s + 1 if s < 5 else 0) for s in range(8)]
    assert out[0][1] == want and out[1][1] == want


def test_survey_shot_list_is_seeded_and_varied():
    import numpy as np
    import bench
    rcv = np.stack(np.meshgrid(np.linspace(0.3, 2.7, 6), np.linspace(0.3, 2.7, 6), [0.01], indexing="ij"), -1).reshape(-1, 3)
    a = bench.survey_shots(4, (3.0, 3.0, 1.5), (8, 8, 4), rcv)
    b = bench.survey_shots(4, (3.0, 3.0, 1.5), (8, 8, 4), rcv)
    assert all(np.array_equal(x["x0"], y["x0"]) and np.array_equal(x["receivers"], y["receivers"]) for x, y in zip(a, b))
    assert len({tuple(x["x0"]) for x in a}) == 4
    assert all(0 < x["x0"][0] < 3.0 for x in a) and all(len(x["receivers"]) == 12 for x in a)
    assert bench.shots_of_rank(7, 1, 3) == [1, 4]
