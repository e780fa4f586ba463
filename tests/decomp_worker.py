"""Worker of tests/test_decomp.py::test_one_process_per_sub_domain: one torch.distributed rank = one sub-domain, all ranks
on cuda:0 (this pool grants one GPU), neighbours' trace buffers mapped through CUDA IPC."""
import os
import sys

import numpy as np


def run(rank, world, port, N, precision, nsteps, hexes, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    here = os.path.dirname(os.path.abspath(__file__))
    sys.path.insert(0, os.path.dirname(here))
    from workloads import make_config
    from paper_1506_00907_b200.decomp import RankDecomposition, partition_elements
    cfg = make_config("cfg2_two_layer", hexes=hexes, N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    part = partition_elements(cfg["EToV"], cfg["VX"], world)
    dd = RankDecomposition(dist, N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part,
                           default_bc=cfg["default_bc"])
    torch.cuda.set_device(0)
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    dd.dg_step(nsteps)
    q = dd.dg_get_fields()
    if rank == 0:
        np.save(out_path, q)
    dist.barrier()
    dd.close()
    dist.destroy_process_group()
