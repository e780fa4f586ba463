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
@pytest.mark.parametrize("N,precision,nparts,fused", [(3, 32, 2, False), (3, 64, 3, False), (4, 32, 3, False), (2, 64, 4, False),
                                                      (3, 32, 3, True), (3, 64, 2, True), (4, 64, 2, True), (1, 64, 3, True),
                                                      (5, 64, 2, True)])
def test_decomposed_run_matches_the_oracle(N, precision, nparts, fused):
    """fused: no k_halo launches - the step kernel (k_pipe; k_step at N = 1 and N = 5 fp64) reads the exterior states of
    the halo faces from the neighbour's trace buffer itself (dg_halo_sources)."""
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    cfg = _cfg(N=N)
    nsteps = cfg["nsteps"]
    part = partition_elements(cfg["EToV"], cfg["VX"], nparts)
    dd = Decomposition(N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"],
                       fused=fused)
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    n0 = dd.launch_count()
    dd.dg_step(nsteps)
    q = dd.dg_get_fields()
    if fused:
        assert dd.launch_count() - n0 == nsteps * nparts             # one launch per sub-domain and time step: the step kernel
    else:
        assert dd.launch_count() - n0 >= nsteps * nparts * 2         # a halo fetch and a step per sub-domain and time step
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


def _lts_cfg(N, hexes=(6, 6, 8), nsteps=100):
    cfg = make_config("cfg3_lts", hexes=hexes, N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    return cfg


def test_multirate_halo_sets_carry_one_level_each():
    """Host logic of the multi-rate decomposition: the sub-domains take the levels of the whole mesh (also where a part
    alone would grade differently), weights 2^l balance the local steps, every halo set points at elements
    of ONE level of the neighbour, and an element whose finer neighbour lies across the cut is laid out among the
    elements that expose half-step traces (first slots of its level)."""
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    import paper_1506_00907_b200 as pk
    cfg = _lts_cfg(2)
    g = pk.DG(cfg["N"], 64, cfg["EToV"], cfg["VX"], default_bc=cfg["default_bc"])
    g.dg_set_model(cfg["rho"], cfg["c"], cfg["nlevels"], cfg["cfl"])
    level, EToE = g.dg_get_levels(), g.dg_get_connectivity()[0]
    g.close()
    assert len(np.unique(level)) == 3
    part = partition_elements(cfg["EToV"], cfg["VX"], 3, 2.0 ** level)
    work = np.array([(2.0 ** level[part == p]).sum() for p in range(3)])
    assert work.max() / work.mean() < 1.1, work
    dd = Decomposition(cfg["N"], 64, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"],
                       nlevels=3, cfl=cfg["cfl"])
    cross = 0
    for p, s in enumerate(dd.sub):
        assert np.array_equal(s.dg_get_levels(), level[dd.elems[p]])
        assert s.dg_get_dt() == (dd.dt, 4)                             # the finest step of the whole mesh, 2^(L-1) per global step
        slots = [x.dg_get_slots() for x in dd.sub]
        bk, bf, bc = s.dg_get_boundary_faces()
        for i, (q, bnd, rec, pos) in enumerate(dd.sets[p]):
            lev = dd.set_level[p][i]
            behind = {int(sl): k for k, sl in enumerate(slots[q])}
            for h in range(bnd.size):
                assert level[dd.elems[q][behind[int(rec[h] // 4)]]] == lev
                mine = level[dd.elems[p][bk[bnd[h]]]]
                assert abs(int(mine) - lev) <= 1
                cross += mine != lev
        # elements with a finer neighbour, inside or across the cut, come first within their level
        sl = s.dg_get_slots()
        for lev in range(3):
            e = dd.elems[p][level[dd.elems[p]] == lev]
            if e.size == 0:
                continue
            nbl = np.where(EToE[e] >= 0, level[np.maximum(EToE[e], 0)], -1)
            finer = (nbl > lev).any(axis=1)
            order = np.argsort(sl[dd.local[e]])
            assert not np.any(np.diff(finer[order].astype(int)) > 0)       # all True, then all False
    assert cross > 0                                                   # the cuts do cross level interfaces
    dd.close()
    # finest-level elements lumped with their neighbours before the bisection: none of their faces is cut,
    # the weights stay balanced
    from paper_1506_00907_b200.decomp import face_neighbours
    assert np.array_equal(np.sort(face_neighbours(cfg["EToV"]), axis=1), np.sort(EToE, axis=1))
    cut_faces = lambda part: sum(1 for k in np.nonzero(level == 2)[0] for k2 in EToE[k] if k2 >= 0 and part[k2] != part[k])
    plain = partition_elements(cfg["EToV"], cfg["VX"], 5, 2.0 ** level)
    lumped = partition_elements(cfg["EToV"], cfg["VX"], 5, 2.0 ** level, lump=level == 2)
    assert cut_faces(plain) > 0 and cut_faces(lumped) == 0
    work = np.array([(2.0 ** level[lumped == p]).sum() for p in range(5)])
    assert work.max() / work.mean() < 1.1, work


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,nparts,lump,fused", [(3, 64, 2, False, False), (2, 64, 5, False, False),
                                                           (2, 64, 5, True, False), (3, 32, 3, True, False),
                                                           (4, 32, 2, False, False), (3, 64, 3, False, True),
                                                           (4, 32, 5, True, True), (2, 32, 4, False, True)])
def test_decomposed_multirate_run_matches_the_oracle(N, precision, nparts, lump, fused):
    """Three levels, cuts across level interfaces: before every FINE step each sub-domain fetches, per halo set, the
    neighbour's traces of that set's level - its current ones if the level starts a step there, its half-step ones (eq (19))
    if it is in mid-step - and advances by dg_step_fine(1).  Same fields as the single-domain oracle and library runs."""
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    cfg = _lts_cfg(N)
    nsteps = cfg["nsteps"]
    o = make_oracle(cfg)
    part = partition_elements(cfg["EToV"], cfg["VX"], nparts, 2.0 ** np.asarray(o.level),
                              lump=(np.asarray(o.level) == 2) if lump else None)
    dd = Decomposition(N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"],
                       nlevels=cfg["nlevels"], cfl=cfg["cfl"], fused=fused)
    assert np.array_equal(dd.level, o.level)
    assert any(dd.set_level[p][i] != lev for p in range(nparts) for i, (q, bnd, _, _) in enumerate(dd.sets[p])
               for lev in dd.level[dd.elems[p][dd.sub[p].dg_get_boundary_faces()[0][bnd]]])
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    dd.dg_step(nsteps)
    q = dd.dg_get_fields()
    assert fused or (dd.pulls[0] > 0 and dd.pulls[2] > 0)
    if fused:
        assert dd.pulls.sum() == 0                                     # no fetch launches at all
    elif lump:                                                           # the finest level is off the cuts: the fine steps that
        assert dd.pulls[1] == 0 and dd.pulls[3] == 0                   # advance it alone exchange nothing
    elif nparts == 5:
        assert dd.pulls[1] > 0 and dd.pulls[3] > 0
    dd.close()
    F = o.new_field()
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    share = np.array([np.linalg.norm(F.q[part == p]) for p in range(nparts)]) / np.linalg.norm(F.q)
    assert share.min() > 0.005, share                                  # the wave has crossed every cut
    assert rel_l2(q, F.q) < (1e-10 if precision == 64 else 1e-5), rel_l2(q, F.q)
    g = make_gpu(cfg, precision)
    g.dg_step(nsteps)
    q1 = g.dg_get_fields()
    g.close()
    assert rel_l2(q, q1) < (1e-13 if precision == 64 else 2e-6), rel_l2(q, q1)


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,nparts,nlevels", [(3, 64, 2, 1), (3, 32, 3, 1), (2, 64, 3, 3), (4, 32, 2, 3), (3, 64, 4, 3),
                                                        (1, 64, 3, 3), (5, 64, 2, 1)])      # the last two: k_step, two fields
def test_rtm_shot_on_a_decomposed_mesh(N, precision, nparts, nlevels):
    """Both phases of a shot with the mesh cut into sub-domains: every sub-domain captures and replays the
    traces of its own absorbing faces, records and injects at its own receivers, keeps its part of the image; the source
    and - backward - the receiver wavefield exchange halo traces inside the step kernels before every fine step
    (rtm_forward_part / rtm_backward_part, dg_halo_sources / rtm_halo_sources).  Signals, final state and image equal
    the single-domain oracle's."""
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    nsteps = 60 if nlevels == 1 else 32
    if nlevels == 1:
        cfg = make_config("cfg4_rtm", hexes=(5, 5, 3), N=N, nsteps=nsteps, n_receivers_side=4)
    else:
        cfg = make_config("cfg3_lts", hexes=(5, 5, 6), N=N, nsteps=nsteps)
        gx = np.linspace(0.4, 2.6, 4)
        cfg["receivers"] = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
        cfg["updir"] = np.array([0.0, 0.0, -1.0])
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    lev = np.asarray(o.level)
    part = partition_elements(cfg["EToV"], cfg["VX"], nparts, 2.0 ** lev)
    dd = Decomposition(N, precision, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"],
                       nlevels=nlevels, cfl=cfg["cfl"], fused=True)
    dd.bind_torch("cuda:0")
    s = cfg["source"]
    dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    dd.rtm_bind(nsteps, cfg["receivers"], "cuda:0")
    assert sum(sel.size > 0 for sel in dd.rcv_sel) >= 2              # the receivers lie in several sub-domains
    tol = 1e-10 if precision == 64 else 1e-5
    data_g = dd.rtm_forward_shot(nsteps)
    data_o, hist, qT = o.rtm_forward(nsteps)
    assert np.abs(data_o).max() > 0
    assert rel_l2(data_g, data_o) < tol, rel_l2(data_g, data_o)
    assert rel_l2(dd.dg_get_fields(), qT) < tol
    share_q = np.array([np.linalg.norm(qT[part == p]) for p in range(nparts)]) / np.linalg.norm(qT)
    assert share_q.min() > 1e-3, share_q                              # the wave has crossed every cut
    dd.rtm_backward_shot(nsteps, data_o, updir=tuple(cfg["updir"]))
    I_o, FS, FR = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], nglobal_total=nsteps)
    img = dd.rtm_image_read()
    share = np.array([np.linalg.norm(I_o[part == p]) for p in range(nparts)]) / np.linalg.norm(I_o)
    assert np.abs(I_o).max() > 0 and (share > 1e-6).sum() >= 2, share
    assert rel_l2(img, I_o) < (1e-4 if precision == 32 else 1e-10), rel_l2(img, I_o)
    dd.close()


@pytest.mark.gpu
@pytest.mark.parametrize("nlevels,window", [(1, 4), (3, 2)])
def test_decomposed_rtm_shot_with_spilled_traces_is_bit_identical(nlevels, window):
    """The shot in parts on sub-domains whose trace histories live in pinned host memory behind a small device ring
    (rtm_set_trace_spill): capture copies follow the parts, replay fetches run ahead of them; same bits as in HBM."""
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements
    nsteps, N, nparts = 24, 3, 3
    if nlevels == 1:
        cfg = make_config("cfg4_rtm", hexes=(5, 5, 3), N=N, nsteps=nsteps, n_receivers_side=4)
    else:
        cfg = make_config("cfg3_lts", hexes=(5, 5, 6), N=N, nsteps=nsteps)
        gx = np.linspace(0.4, 2.6, 4)
        cfg["receivers"] = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    part = partition_elements(cfg["EToV"], cfg["VX"], nparts)
    res = []
    for w in (0, window):
        dd = Decomposition(N, 32, cfg["EToV"], cfg["VX"], cfg["rho"], cfg["c"], part, default_bc=cfg["default_bc"],
                           nlevels=nlevels, cfl=cfg["cfl"], fused=True)
        dd.bind_torch("cuda:0")
        s = cfg["source"]
        dd.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
        dd.rtm_bind(nsteps, cfg["receivers"], "cuda:0", spill_window=w)
        data = dd.rtm_forward_shot(nsteps)
        dd.rtm_backward_shot(nsteps, data)
        res.append((data, dd.rtm_image_read()))
        dd.close()
    assert np.abs(res[0][1]).max() > 0
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


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
        g.dg_get_trace_device()                                      # one buffer only for single-rate: dg_get_trace_levels
    cur, half, n = g.dg_get_trace_levels()
    assert len(cur) == 3 and half not in cur and n > 0
    g.dg_step_fine(1)
    with pytest.raises(pk.DGError):
        g.dg_step(1)                                                 # inside a global step
    g.dg_step_fine(3)
    g.dg_step(1)
    lev = g.dg_get_levels()
    with pytest.raises(pk.DGError):
        g.dg_set_model_levels(cfg3["rho"], cfg3["c"], 3, 1e-4, np.where(lev == 1, 3, lev))     # level out of range
    with pytest.raises(pk.DGError):
        g.dg_set_model_levels(cfg3["rho"], cfg3["c"], 3, 1e-4, np.where(lev == 1, 0, lev))     # neighbours two levels apart
    g.close()
    # fused exchange and shot phases in parts: one fine step per set of sources, parts in order
    g = make_gpu(cfg3, 64, history_steps=4)
    g.dg_halo_sources([])                                            # no halo sets: nothing to name
    with pytest.raises(pk.DGError) as e:
        g.dg_step(1)                                                 # 4 fine steps on sources good for one
    assert e.value.code == pk.DG_ERR_STATE
    g.dg_step_fine(1)                                                # the failed call did not consume them ... and this one does
    g.dg_step_fine(3)
    with pytest.raises(pk.DGError):
        g.rtm_forward_part(4, 3, 1)                                  # a phase starts at fine step 0
    g.rtm_forward_part(4, 0, 5)
    with pytest.raises(pk.DGError):
        g.rtm_forward_part(4, 4, 1)                                  # parts follow one another
    with pytest.raises(pk.DGError):
        g.rtm_backward_part(4, None, 0, 1)                           # no finished forward phase
    g.rtm_forward_part(4, 5, 11)
    g.rtm_backward_part(4, None, 0, 0)
    with pytest.raises(pk.DGError):
        g.rtm_backward_part(4, None, 2, 1)
    with pytest.raises(pk.DGError):
        g.rtm_backward_part(4, None, 0, 17)                          # beyond the phase
    g.rtm_backward_part(4, None, 0, 16)
    with pytest.raises(pk.DGError):
        g.rtm_get_trace_levels(2)
    g.dg_set_integrator(pk.DG_INTEGRATOR_AB3)
    g.close()
    g1 = make_gpu(_cfg(hexes=(3, 3, 2)), 64)
    g1.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
    with pytest.raises(pk.DGError) as e:
        g1.dg_halo_sources([])                                       # the fused exchange is in the AB step kernels
    assert e.value.code == pk.DG_ERR_UNSUPPORTED
    g1.close()


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,world,workload,fused", [(3, 64, 2, "cfg2_two_layer", False), (3, 32, 3, "cfg2_two_layer", False),
                                                              (3, 64, 3, "cfg3_lts", False), (3, 64, 3, "cfg3_lts", True),
                                                              (4, 32, 2, "cfg2_two_layer", True)])
def test_one_process_per_sub_domain(N, precision, world, workload, fused, tmp_path):
    """RankDecomposition: one process per sub-domain (gloo for the host side, CUDA IPC mappings of the neighbours'
    workspaces as the source of k_halo), all on cuda:0 here.  Same result as the single-domain run of the library."""
    import socket
    import torch.multiprocessing as mp
    import decomp_worker
    nsteps, hexes = (60, (6, 5, 4)) if workload == "cfg2_two_layer" else (50, (6, 6, 8))   # cfg3_lts: three levels
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "q.npy")
    mp.spawn(decomp_worker.run, args=(world, port, N, precision, nsteps, hexes, out, workload, fused), nprocs=world, join=True)
    q = np.load(out)
    cfg = _cfg(hexes=hexes, N=N) if workload == "cfg2_two_layer" else _lts_cfg(N, hexes=hexes, nsteps=nsteps)
    g = make_gpu(cfg, precision)
    g.dg_step(nsteps)
    q1 = g.dg_get_fields()
    g.close()
    assert np.linalg.norm(q1) > 0
    assert rel_l2(q, q1) < (1e-13 if precision == 64 else 2e-6), rel_l2(q, q1)


@pytest.mark.gpu
@pytest.mark.parametrize("N,precision,world,workload", [(3, 64, 2, "cfg2_two_layer"), (2, 64, 3, "cfg3_lts")])
def test_rtm_shot_one_process_per_sub_domain(N, precision, world, workload, tmp_path):
    """The whole shot with one process per sub-domain: the step kernels of a rank read both wavefields' halo traces from
    the CUDA-IPC mappings of its neighbours' workspace (source field) and RTM region (receiver field).  Same signals,
    final state and image as the single-domain run of the library."""
    import socket
    import torch.multiprocessing as mp
    import decomp_worker
    nsteps, hexes = (40, (6, 5, 4)) if workload == "cfg2_two_layer" else (24, (5, 5, 6))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "shot.npz")
    mp.spawn(decomp_worker.run_rtm, args=(world, port, N, precision, nsteps, hexes, out, workload), nprocs=world, join=True)
    res = np.load(out)
    cfg = make_config(workload, hexes=hexes, N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    gx = np.linspace(0.4, 2.6, 4)
    cfg["receivers"] = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
    g = make_gpu(cfg, precision, history_steps=nsteps)
    data = g.rtm_forward_shot(nsteps)
    qT = g.rtm_get_fields(0)
    g.rtm_backward_shot(nsteps, data, updir=(0.0, 0.0, -1.0))
    img = g.rtm_image_read()
    g.close()
    assert np.abs(data).max() > 0 and np.abs(img).max() > 0
    assert rel_l2(res["data"], data) < 1e-12 and rel_l2(res["qT"], qT) < 1e-12
    assert rel_l2(res["img"], img) < 1e-11, rel_l2(res["img"], img)


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
