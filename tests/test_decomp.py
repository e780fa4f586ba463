"""Domain decomposition (paper_1506_00907_b200/decomp.py).

CPU (host logic): the weighted partition balances the weights; every halo face of every sub-domain points at the record
of the SAME geometric face in its neighbour, node by node (physical coordinates of my face node i and of the neighbour's
node src_pos[i] coincide), and every cut face of the mesh is a halo face on both sides.

GPU: the decomposed run - exterior states of the cut faces fetched on the device from the neighbour's trace buffer by
k_halo before every step - reproduces the single-domain oracle within the north_star tolerances, and the single-domain
run of the library to rounding: the flux across a cut uses the same traces and the same single-valued impedance
(reading Q4, dg_set_exterior_impedance) as the interior face it replaces."""
import numpy as np
import pytest

from workloads import make_config
from parity_util import make_oracle, make_gpu, rel_l2


def _nodes_xyz(g, etov, vx):
    """Physical coordinates of every node of every element [K][Np][3] from the reference nodes (affine map)."""
    r, s, t = g.dg_get_nodes()
    v = vx[etov]                                                     # [K][4][3]
    L = np.stack([-(1 + r + s + t) / 2, (1 + r) / 2, (1 + s) / 2, (1 + t) / 2], axis=1)   # [Np][4]
    return np.einsum("nv,kvd->knd", L, v)


def _cfg(hexes=(6, 5, 4), N=3):
    cfg = make_config("cfg2_two_layer", hexes=hexes, N=N, nsteps=120)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    return cfg


@pytest.mark.parametrize("nparts", [2, 3, 5])
def test_partition_and_halo_tables(nparts):
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    cfg = _cfg()
    etov, vx = cfg["EToV"], cfg["VX"]
    rng = np.random.default_rng(7)
    w = rng.choice([1.0, 2.0, 4.0], size=etov.shape[0], p=[0.7, 0.25, 0.05])      # local steps per global step
    part = partition_elements(etov, vx, nparts, w)
    sums = np.array([w[part == p].sum() for p in range(nparts)])
    assert part.min() == 0 and part.max() == nparts - 1
    assert sums.max() / sums.mean() < 1.15, sums                     # balanced in weight, not in count
    dd = Decomposition(cfg["N"], 64, etov, vx, cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"])
    Fmask = dd.sub[0].dg_get_operators()[4]
    xyz = [_nodes_xyz(s, s_etov, s_vx) for s, s_etov, s_vx in
           ((dd.sub[p], *_local_mesh(etov, vx, dd.elems[p])) for p in range(nparts))]
    slots = [s.dg_get_slots() for s in dd.sub]
    ncut = 0
    for p in range(nparts):
        bk, bf, bc = dd.sub[p].dg_get_boundary_faces()
        seen = np.zeros(bk.size, dtype=bool)
        for q, bnd, rec, pos in dd.sets[p]:
            slot_to_elem = {int(sl): k for k, sl in enumerate(slots[q])}
            for h in range(bnd.size):
                k, f = int(bk[bnd[h]]), int(bf[bnd[h]])
                k2, f2 = slot_to_elem[int(rec[h] // 4)], int(rec[h] % 4)
                mine = xyz[p][k][Fmask[f]]
                theirs = xyz[q][k2][Fmask[f2]][pos[h]]
                assert np.abs(mine - theirs).max() < 1e-12
                seen[bnd[h]] = True
                ncut += 1
        assert np.array_equal(seen, bc == 4)                          # every prescribed face here is a halo face
    # every cut face of the mesh appears once from each side
    g = dd.sub[0].__class__(cfg["N"], 64, etov, vx, default_bc=cfg["default_bc"])
    EToE = g.dg_get_connectivity()[0]
    g.close()
    ncut_mesh = int(((EToE >= 0) & (part[np.maximum(EToE, 0)] != part[:, None])).sum())
    assert ncut == ncut_mesh and ncut > 0
    dd.close()


def _local_mesh(etov, vx, elems):
    verts, inv = np.unique(etov[elems], return_inverse=True)
    return inv.reshape(-1, 4).astype(np.int32), vx[verts]


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,nparts", [(3, 32, 2), (3, 64, 3), (4, 32, 3), (2, 64, 4)])
def test_decomposed_run_matches_the_oracle(N, precision, nparts):
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    cfg = _cfg(N=N)
    nsteps = cfg["nsteps"]
    part = partition_elements(cfg["EToV"], cfg["VX"], nparts)
    dd = Decomposition(N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"])
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    dd.dg_step(nsteps)
    q = dd.dg_get_fields()
    assert dd.launch_count() >= nsteps * nparts * 2                  # a halo fetch and a step per sub-domain and time step
    dd.close()
    o = make_oracle(cfg)
    F = o.new_field()
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    tol = 1e-10 if precision == 64 else 1e-5
    assert rel_l2(q, F.q) < tol, rel_l2(q, F.q)
    g = make_gpu(cfg, precision)
    g.dg_step(nsteps)
    q1 = g.dg_get_fields()
    g.close()
    assert rel_l2(q, q1) < (1e-13 if precision == 64 else 2e-6), rel_l2(q, q1)


@pytest.mark.gpu
def test_halo_and_spill_calls_reject_bad_arguments():
    """Error behaviour stated in include/dgrtm.h: wrong arguments come back as error codes (DGError), nothing aborts."""
    import paper_1506_00907_b200 as pk
    cfg = _cfg(hexes=(3, 3, 2))
    g = make_gpu(cfg, 32)                                            # absorbing faces only: none is DG_BC_PRESCRIBED
    Nfp = g.Nfp
    with pytest.raises(pk.DGError):
        g.dg_set_halo(0, np.array([0]), np.array([0]), np.zeros((1, Nfp), dtype=np.int32))      # not a prescribed face
    with pytest.raises(pk.DGError):
        g.dg_set_halo(9, np.array([0]), np.array([0]), np.zeros((1, Nfp), dtype=np.int32))      # set out of range
    with pytest.raises(pk.DGError):
        g.dg_halo_pull(0, 0)                                         # NULL source
    with pytest.raises(pk.DGError):
        g.rtm_set_trace_spill(1 << 20, 4096, 1)                      # window < 2
    g.close()
    cfg3 = make_config("cfg3_lts", hexes=(4, 4, 6), N=2)
    g = make_gpu(cfg3, 32)
    with pytest.raises(pk.DGError):
        g.dg_get_trace_device()                                      # the halo exchange is single-rate
    g.close()


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,world", [(3, 64, 2), (3, 32, 3)])
def test_one_process_per_sub_domain(N, precision, world, tmp_path):
    """RankDecomposition: one process per sub-domain (gloo for the host side, CUDA IPC mappings of the neighbours'
    workspaces as the source of k_halo), all on cuda:0 here.  Same result as the single-domain run of the library."""
    import socket
    import torch.multiprocessing as mp
    import decomp_worker
    nsteps, hexes = 60, (6, 5, 4)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "q.npy")
    mp.spawn(decomp_worker.run, args=(world, port, N, precision, nsteps, hexes, out), nprocs=world, join=True)
    q = np.load(out)
    cfg = _cfg(hexes=hexes, N=N)
    g = make_gpu(cfg, precision)
    g.dg_step(nsteps)
    q1 = g.dg_get_fields()
    g.close()
    assert np.linalg.norm(q1) > 0
    assert rel_l2(q, q1) < (1e-13 if precision == 64 else 2e-6), rel_l2(q, q1)


@pytest.mark.parametrize("world", [2, 3])
def test_rank_decomposition_plan_gloo(world, tmp_path):
    """The N > 1 path on the CPU (gloo, world size 2 and 3): every rank's halo requests, answered by the neighbour from its
    own sub-domain alone, are the coordinates of the requester's halo face nodes (tests/decomp_worker.py::check_plan)."""
    import socket
    import torch.multiprocessing as mp
    import decomp_worker
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "plan.npy")
    mp.spawn(decomp_worker.check_plan, args=(world, port, 3, (5, 4, 3), out), nprocs=world, join=True)
    res = np.load(out)
    assert res.shape == (world, 2) and res[:, 1].min() > 0           # every rank has halo faces
    assert res[:, 0].max() < 1e-12
