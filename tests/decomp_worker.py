"""Worker of tests/test_decomp.py::test_one_process_per_sub_domain: one torch.distributed rank = one sub-domain, all ranks
on cuda:0 (this pool grants one GPU), neighbours' trace buffers mapped through CUDA IPC."""
import os
import sys

import numpy as np


def run(rank, world, port, N, precision, nsteps, hexes, out_path, workload="cfg2_two_layer", fused=False):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    here = os.path.dirname(os.path.abspath(__file__))
    sys.path.insert(0, os.path.dirname(here))
    from workloads import make_config
    from paper_1506_00907_b200.decomp import RankDecomposition, partition_elements
    cfg = make_config(workload, hexes=hexes, N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    part = partition_elements(cfg["EToV"], cfg["VX"], world)
    dd = RankDecomposition(dist, N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part,
                           default_bc=cfg["default_bc"], nlevels=cfg["nlevels"], cfl=cfg["cfl"], fused=fused)
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


def run_rtm(rank, world, port, N, precision, nsteps, hexes, out_path, workload):
    """A whole RTM shot with one process per sub-domain: rank 0 saves the recorded signals, the final state and the image."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    here = os.path.dirname(os.path.abspath(__file__))
    sys.path.insert(0, os.path.dirname(here))
    from workloads import make_config
    from paper_1506_00907_b200.decomp import RankDecomposition, partition_elements
    cfg = make_config(workload, hexes=hexes, N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    gx = np.linspace(0.4, 2.6, 4)
    xr = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
    part = partition_elements(cfg["EToV"], cfg["VX"], world)
    dd = RankDecomposition(dist, N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part,
                           default_bc=cfg["default_bc"], nlevels=cfg["nlevels"], cfl=cfg["cfl"], fused=True)
    torch.cuda.set_device(0)
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    dd.rtm_bind(nsteps, xr, "cuda:0")
    data = dd.rtm_forward_shot(nsteps)
    qT = dd.dg_get_fields()
    dd.rtm_backward_shot(nsteps, data, updir=(0.0, 0.0, -1.0))
    img = dd.rtm_image_read()
    if rank == 0:
        np.savez(out_path, data=data, qT=qT, img=img)
    dist.barrier()
    dd.close()
    dist.destroy_process_group()


def check_plan(rank, world, port, N, hexes, out_path):
    """CPU (gloo) check of the one-process-per-sub-domain plan: every rank asks each neighbour - which answers from its OWN
    sub-domain only - for the physical coordinates of the trace-record entries it is going to read, and compares them
    with the coordinates of its own halo face nodes."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import torch.distributed as dist
    dist.init_process_group("gloo", rank=rank, world_size=world)
    here = os.path.dirname(os.path.abspath(__file__))
    sys.path.insert(0, os.path.dirname(here))
    from workloads import make_config
    from paper_1506_00907_b200.decomp import RankDecomposition, partition_elements
    cfg = make_config("cfg2_two_layer", hexes=hexes, N=N)
    etov, vx = cfg["EToV"], cfg["VX"]
    part = partition_elements(etov, vx, world)
    dd = RankDecomposition(dist, N, 64, etov, vx, cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"])
    me = dd.sub[rank]

    def node_xyz(elems_global):
        r, s, t = me.dg_get_nodes()
        L = np.stack([-(1 + r + s + t) / 2, (1 + r) / 2, (1 + s) / 2, (1 + t) / 2], axis=1)
        return np.einsum("nv,kvd->knd", L, vx[etov[elems_global]])

    Fmask = me.dg_get_operators()[4]
    mine_xyz = node_xyz(dd.elems[rank])                               # [Kp][Np][3] of MY elements
    slot_to_elem = np.argsort(me.dg_get_slots())                      # my slots are a permutation of 0..Kp-1 plus padding
    slots = me.dg_get_slots()
    lookup = {int(sl): k for k, sl in enumerate(slots)}
    requests = [None] * world
    dist.all_gather_object(requests, {q: (rec, pos) for q, _, rec, pos in dd.sets[rank]})
    answers = {}
    for p in range(world):                                            # what rank p wants to read from MY buffer
        if p != rank and rank in requests[p]:
            rec, pos = requests[p][rank]
            k = np.array([lookup[int(x)] for x in rec // 4])
            f = (rec % 4).astype(int)
            answers[p] = np.stack([mine_xyz[k[h]][Fmask[f[h]]][pos[h]] for h in range(len(rec))])
    replies = [None] * world
    dist.all_gather_object(replies, answers)
    bk, bf, _ = me.dg_get_boundary_faces()
    worst, n = 0.0, 0
    for q, bnd, rec, pos in dd.sets[rank]:
        theirs = replies[q][rank]
        for h in range(len(bnd)):
            own = mine_xyz[bk[bnd[h]]][Fmask[bf[bnd[h]]]]
            worst = max(worst, float(np.abs(own - theirs[h]).max()))
            n += 1
    res = [None] * world
    dist.all_gather_object(res, (worst, n))
    if rank == 0:
        np.save(out_path, np.array(res))
    dist.barrier()
    dd.close()
    dist.destroy_process_group()
