"""Parity of the CUDA path (through the C ABI of include/dgrtm.h) with the fp64 oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star's: bit-exact for
connectivity, levels and trace indexing; relative L2 <= 1e-10 (fp64) / 1e-5 (fp32) for fields after
the stated step counts; image relative L2 <= 1e-4 in fp32.

Sizes: meshes the oracle finishes in seconds that still span several 32-element blocks and a ragged
last block (K = 6*nx*ny*nz is never a multiple of 32 for the odd sizes used)."""
import numpy as np
import pytest

from workloads import box_tet_mesh, graded_box_tet_mesh, make_config, permute_elements
from parity_util import make_oracle, make_gpu, rel_l2, cavity_mode, random_state

pytestmark = pytest.mark.gpu

TOL = {64: 1e-10, 32: 1e-5}
TOL_RHS = {64: 1e-12, 32: 2e-6}          # one operator application (no accumulation over steps)


def _mixed_bc_cfg(N, hexes=(3, 3, 2), seed=21):
    """Small jittered box with all four boundary types (one per side group) and random material."""
    etov, vx = box_tet_mesh(*hexes, lengths=(1.5, 1.5, 1.0), jitter=0.1, seed=seed)
    etov, _ = permute_elements(etov, seed + 1)
    K = etov.shape[0]
    rng = np.random.default_rng(seed)
    cen = vx[etov].mean(axis=1)
    face_bc = np.zeros((K, 4), dtype=np.int8)
    # by element centroid octant: type 1..4 (entries of interior faces are ignored)
    face_bc[:] = (1 + (cen[:, 0] > 0.75).astype(int) + 2 * (cen[:, 1] > 0.75).astype(int))[:, None]
    cfg = dict(EToV=etov, VX=vx, rho=rng.uniform(1.0, 2.5, K), c=rng.uniform(1.5, 4.5, K), N=N,
               precision=64, default_bc=2, nlevels=1, cfl=0.15, source=None, receivers=None)
    return cfg, face_bc


# ---------------------------------------------------------------------------------------------------
# S0 setup: bit-exact integers, fp64 tables
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6])
def test_setup_tables(N):
    cfg, face_bc = _mixed_bc_cfg(N)
    o = make_oracle(cfg, face_bc=face_bc)
    g = make_gpu(cfg, 64, face_bc=face_bc)
    r, s, t = g.dg_get_nodes()
    assert np.abs(r - o.ref.r).max() < 1e-13 and np.abs(s - o.ref.s).max() < 1e-13 and np.abs(t - o.ref.t).max() < 1e-13
    Dr, Ds, Dt, LIFT, Fmask = g.dg_get_operators()
    assert np.array_equal(Fmask, o.ref.Fmask)
    for a, b in ((Dr, o.ref.Dr), (Ds, o.ref.Ds), (Dt, o.ref.Dt), (LIFT, o.ref.LIFT)):
        assert np.abs(a - b).max() < 1e-10 * max(1.0, np.abs(b).max())
    EToE, EToF, mapP = g.dg_get_connectivity()
    assert np.array_equal(EToE, o.EToE) and np.array_equal(EToF, o.EToF)
    interior = o.EToE >= 0
    assert np.array_equal(mapP[interior], o.mapP[interior])
    bk, bf, bc = g.dg_get_boundary_faces()
    assert np.array_equal(bk, o.bnd_k) and np.array_equal(bf, o.bnd_f)
    assert np.array_equal(bc, o.bc[o.bnd_k, o.bnd_f])
    geo = g.dg_get_geometry()
    for key in ("J", "ginv", "normals", "gsur", "ell"):
        assert np.abs(geo[key] - o.geo[key]).max() < 1e-12 * np.abs(o.geo[key]).max(), key
    dt, nloc = g.dg_get_dt()
    assert abs(dt - o.dt_local) < 1e-15 * o.dt_local and nloc == o.nlocal
    g.close()


def test_levels_and_point_terms_bit_exact():
    cfg = make_config("cfg3_lts", hexes=(6, 6, 8), N=2)
    cfg["receivers"] = np.array([[0.31, 0.42, 0.11], [1.7, 2.2, 0.9], [2.9, 0.1, 1.4]])
    o = make_oracle(cfg)
    g = make_gpu(cfg, 64)
    lv = g.dg_get_levels()
    assert np.array_equal(lv, o.level)
    assert len(np.unique(lv)) == 3, "the workload must populate all three levels"
    k, w = g.dg_get_source()
    assert k == o.source["k"] and np.abs(w - o.source["w"]).max() < 1e-10 * np.abs(w).max()
    rk, rows, rw = g.dg_get_receivers()
    assert np.array_equal(rk, o.receivers["k"])
    assert np.abs(rows - o.receivers["row"]).max() < 1e-11
    assert np.abs(rw - o.receivers["w"]).max() < 1e-10 * np.abs(rw).max()
    g.close()


# ---------------------------------------------------------------------------------------------------
# S1 volume / S2 surface: one application on a random state, every order, both precisions
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6])
def test_rhs_volume_surface(N, precision):
    cfg, face_bc = _mixed_bc_cfg(N)
    o = make_oracle(cfg, face_bc=face_bc)
    g = make_gpu(cfg, precision, face_bc=face_bc)
    q = random_state(o.K, o.Np, 100 + N)
    rng = np.random.default_rng(7)
    ext = rng.standard_normal((o.bnd_k.size, o.Nfp, 2))
    g.dg_set_state(q)
    g.dg_set_exterior(ext)
    F = o.new_field(q)
    qf = g.dg_get_traces()
    assert rel_l2(qf, F.qf) < TOL_RHS[precision]
    # exterior applies to prescribed faces only here (absorbing faces: exterior = 0)
    presc = o.bc[o.bnd_k, o.bnd_f] == 4
    ext_o = np.where(presc[:, None, None], ext, 0.0)
    rv = o.rhs_volume(F.q)
    assert rel_l2(g.dg_get_rhs(0, 1), rv) < TOL_RHS[precision]
    for direction in (1, -1):
        rs = o.rhs_surface(F.q, F.qf, direction=direction, exterior=ext_o)
        assert rel_l2(g.dg_get_rhs(1, direction), rs) < TOL_RHS[precision]
        assert rel_l2(g.dg_get_rhs(2, direction), rv + rs) < TOL_RHS[precision]
    g.close()


# ---------------------------------------------------------------------------------------------------
# config 1: cavity mode, fp64, LSERK4 (and AB3), 100 steps
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("integrator", ["lserk4", "ab3"])
def test_cfg1_cavity(integrator):
    import paper_1506_00907_b200 as pk
    cfg = make_config("cfg1_cavity")
    if integrator == "ab3":
        cfg["cfl"] = 0.15
    o = make_oracle(cfg)
    g = make_gpu(cfg, 64)
    q0 = cavity_mode(o.X, 0.0)
    g.dg_set_state(q0)
    F = o.new_field(q0)
    if integrator == "lserk4":
        g.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
        g.dg_step(cfg["nsteps"])
        t_end = o.run_lserk4(F, 0.0, o.dt_local, cfg["nsteps"])
    else:
        g.dg_step(cfg["nsteps"])
        t_end = o.run_mrab([F], cfg["nsteps"], 0.0, 1, source_on=(False,))
    q = g.dg_get_fields()
    assert abs(g.dg_get_time() - t_end) < 1e-12
    assert rel_l2(q, F.q) < TOL[64]
    assert rel_l2(g.dg_get_traces(), F.qf) < TOL[64]
    # closed form: discretisation error only (reported, loose bound)
    assert rel_l2(q, cavity_mode(o.X, t_end)) < 5e-2
    g.close()


# ---------------------------------------------------------------------------------------------------
# config 2 shape: two-layer model, Ricker source, absorbing, single-rate AB3
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,nsteps", [(32, 1000), (64, 300)])
def test_cfg2_two_layer(precision, nsteps):
    cfg = make_config("cfg2_two_layer", hexes=(5, 5, 3), nsteps=nsteps)
    # a source that is already active (the 15 Hz pulse of the config is still ~0 after 1000 tiny steps)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision)
    g.dg_step(nsteps)
    F = o.new_field()
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    q = g.dg_get_fields()
    assert np.linalg.norm(F.q) > 0
    assert rel_l2(q, F.q) < TOL[precision], rel_l2(q, F.q)
    assert per_element_max(q, F.q) < 20 * TOL[precision]
    g.close()


# ---------------------------------------------------------------------------------------------------
# config 3 shape: multi-rate levels 0..2 (Algorithm 1)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,N,nsteps", [(64, 2, 40), (32, 4, 60), (32, 3, 500)])
def test_cfg3_multirate(precision, N, nsteps):
    cfg = make_config("cfg3_lts", hexes=(6, 6, 8), N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    o = make_oracle(cfg)
    assert len(np.unique(o.level)) == 3
    g = make_gpu(cfg, precision)
    assert np.array_equal(g.dg_get_levels(), o.level)
    g.dg_step(nsteps)
    F = o.new_field()
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    assert rel_l2(g.dg_get_fields(), F.q) < TOL[precision]
    assert per_element_max(g.dg_get_fields(), F.q) < 20 * TOL[precision]
    assert rel_l2(g.dg_get_traces(), F.qf) < TOL[precision]
    g.close()


def test_multirate_from_nonzero_state_fp64():
    """AB start-up by AB1, AB2 per element's own steps (reading Q7) under three levels; this mesh
    leaves level 0 EMPTY (degenerate case: a level without elements)."""
    cfg = make_config("cfg3_lts", hexes=(5, 5, 6), N=2, nsteps=7)
    cfg["source"] = None
    o = make_oracle(cfg)
    g = make_gpu(cfg, 64)
    q0 = 1e-3 * random_state(o.K, o.Np, 5)
    g.dg_set_state(q0)
    F = o.new_field(q0)
    g.dg_step(7)
    o.run_mrab([F], 7, 0.0, 1, source_on=(False,))
    assert rel_l2(g.dg_get_fields(), F.q) < TOL[64]
    g.close()


# ---------------------------------------------------------------------------------------------------
# config 4 shape: RTM shot - forward with trace capture, backward with replay + injection + imaging
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision,nlevels,imaging", [(64, 1, 1), (32, 1, 1), (32, 1, 0), (64, 3, 1), (32, 3, 1)])
def test_cfg4_rtm_shot(precision, nlevels, imaging):
    nsteps = 120 if nlevels == 1 else 30
    if nlevels == 1:
        cfg = make_config("cfg4_rtm", hexes=(5, 5, 3), N=3 if precision == 32 else 2, nsteps=nsteps, n_receivers_side=4)
    else:
        cfg = make_config("cfg3_lts", hexes=(6, 6, 8), N=2, nsteps=nsteps)
        gx = np.linspace(0.4, 2.6, 3)
        cfg["receivers"] = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
        cfg["updir"] = np.array([0.0, 0.0, -1.0])
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision, history_steps=nsteps)
    tol = TOL[precision]
    # forward phase
    data_g = g.rtm_forward_shot(nsteps)
    data_o, hist, qT = o.rtm_forward(nsteps)
    assert np.abs(data_o).max() > 0
    assert rel_l2(data_g, data_o) < tol
    assert rel_l2(g.rtm_get_fields(0), qT) < tol
    for l in range(nlevels):
        faces, nrec = g.rtm_get_trace_index(l)
        assert np.array_equal(faces, hist.faces[l])                       # bit-exact indexing
        assert nrec == hist.records[l].shape[0] == nsteps * 2 ** l + 1
        if faces.size == 0:
            continue
        for j in (0, 1, nrec // 2, nrec - 1):
            ref = hist.records[l][j]
            got = g.rtm_get_traces(l, j)
            scale = np.abs(hist.records[l]).max()
            assert np.abs(got - ref).max() <= tol * 10 * scale + 1e-300
    # backward phase on observed data = recorded data of a perturbed run (here: scaled copy, the
    # imaging arithmetic does not care where d_r comes from)
    data = 0.7 * data_o
    nback = nsteps - nsteps // 4
    g.rtm_backward_shot(nback, data, updir=cfg["updir"], imaging=imaging, first_image_step=0)
    I_o, FS, FR = o.rtm_backward(nback, qT, hist, data, updir=cfg["updir"],
                                 mode="characteristic" if imaging else "classical", nglobal_total=nsteps)
    assert rel_l2(g.rtm_get_fields(1), FS.q) < tol * 3
    assert rel_l2(g.rtm_get_fields(2), FR.q) < tol * 3
    I_g = g.rtm_image_read()
    assert np.abs(I_o).max() > 0
    assert rel_l2(I_g, I_o) < (1e-4 if precision == 32 else 1e-10)
    assert per_element_max(I_g, I_o) < (2e-3 if precision == 32 else 1e-9)
    assert per_element_max(g.rtm_get_fields(1), FS.q) < 60 * tol
    # images of successive shots add up; rtm_image_zero clears
    g.rtm_forward_shot(nsteps)
    g.rtm_backward_shot(nback, data, updir=cfg["updir"], imaging=imaging)
    assert rel_l2(g.rtm_image_read(), 2 * I_o) < (1e-4 if precision == 32 else 1e-10)
    g.rtm_image_zero()
    assert np.abs(g.rtm_image_read()).max() == 0
    g.close()


@pytest.mark.parametrize("precision,N,nlevels", [(32, 4, 1), (32, 4, 3), (64, 3, 3), (32, 5, 1), (64, 4, 1), (32, 1, 3),
                                                 (64, 6, 1), (32, 6, 1), (64, 5, 3), (32, 2, 1)])
def test_rtm_shot_other_orders(precision, N, nlevels):
    """The two-wavefield kernels of the other orders / precisions (several warps per element block, padded
    output tiles, imaging scalars in registers, shared or global memory): forward + backward + image."""
    nsteps = 16
    if nlevels == 1:
        cfg = make_config("cfg4_rtm", hexes=(4, 4, 3) if N < 6 else (3, 3, 2), N=N, nsteps=nsteps, n_receivers_side=3)
    else:
        cfg = make_config("cfg3_lts", hexes=(5, 5, 6) if N < 5 else (4, 4, 5), N=N, nsteps=nsteps)
        gx = np.linspace(0.4, 2.6, 3)
        cfg["receivers"] = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
        cfg["updir"] = np.array([0.0, 0.0, -1.0])
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision, history_steps=nsteps)
    tol = TOL[precision]
    data_g = g.rtm_forward_shot(nsteps)
    data_o, hist, qT = o.rtm_forward(nsteps)
    assert np.abs(data_o).max() > 0
    assert rel_l2(data_g, data_o) < tol
    assert rel_l2(g.rtm_get_fields(0), qT) < tol
    g.rtm_backward_shot(nsteps, data_o, updir=cfg["updir"])
    I_o, FS, FR = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], nglobal_total=nsteps)
    assert rel_l2(g.rtm_get_fields(1), FS.q) < tol * 3
    assert rel_l2(g.rtm_get_fields(2), FR.q) < tol * 3
    assert np.abs(I_o).max() > 0
    assert rel_l2(g.rtm_image_read(), I_o) < (1e-4 if precision == 32 else 1e-10)
    g.close()


@pytest.mark.parametrize("imaging,mode", [(2, "classical_trapezoid"), (3, "characteristic_trapezoid")])
@pytest.mark.parametrize("precision,N", [(64, 3), (32, 3), (32, 4), (64, 2)])
def test_rtm_trapezoid_imaging(precision, N, imaging, mode):
    """Imaging with the trapezoid rule (21) instead of the AB-consistent integral (24): SURVEY.md 8(f) item 1."""
    nsteps = 16
    cfg = make_config("cfg4_rtm", hexes=(4, 4, 3), N=N, nsteps=nsteps, n_receivers_side=3)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision, history_steps=nsteps)
    g.rtm_forward_shot(nsteps)
    data_o, hist, qT = o.rtm_forward(nsteps)
    g.rtm_backward_shot(nsteps, data_o, updir=cfg["updir"], imaging=imaging)
    I_o, _, _ = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], mode=mode, nglobal_total=nsteps)
    I_24, _, _ = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], mode=mode.replace("_trapezoid", ""),
                                nglobal_total=nsteps)
    assert np.abs(I_o).max() > 0 and rel_l2(I_o, I_24) > 1e-6          # the two quadratures really differ
    assert rel_l2(g.rtm_image_read(), I_o) < (1e-4 if precision == 32 else 1e-10)
    g.close()


def test_survey_stacks_images_in_the_library():
    """several gathers over one mesh: the set-up (operators, geometry,
    connectivity, levels, device tables) is made once ("preparatory phase ... once for the complete survey",
    PAPER.md:478), source and receiver set change between shots, and the images add up IN the library:
    with a receiver capacity reserved, dg_set_receivers keeps the bound RTM region and its image."""
    nsteps = 24
    cfg = make_config("cfg4_rtm", hexes=(5, 4, 3), N=3, nsteps=nsteps, n_receivers_side=3)
    shots = [dict(x0=cfg["source"]["x0"], rcv=cfg["receivers"]),
             dict(x0=cfg["source"]["x0"] + np.array([0.41, -0.33, 0.05]), rcv=cfg["receivers"][::2] + np.array([0.07, 0.03, 0.0])),
             dict(x0=cfg["source"]["x0"] + np.array([-0.52, 0.27, 0.02]), rcv=cfg["receivers"][1::3] + np.array([-0.05, 0.04, 0.0]))]
    for precision in (64, 32):
        g = make_gpu(cfg, precision)
        g.rtm_set_receiver_capacity(max(len(sh["rcv"]) for sh in shots))
        g.bind_history_torch(nsteps)
        launches0 = g.dg_get_launch_count()
        I_sum = 0.0
        for n, sh in enumerate(shots):
            c2 = dict(cfg, source=dict(cfg["source"], x0=sh["x0"], f0=60.0, tp=0.01), receivers=sh["rcv"])
            o = make_oracle(c2)
            data_o, hist, qT = o.rtm_forward(nsteps)
            I_o, _, _ = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], nglobal_total=nsteps)
            I_sum = I_sum + I_o
            before = g.rtm_image_read()
            g.dg_set_source(sh["x0"], 60.0, 0.01, 1.0)
            g.dg_set_receivers(sh["rcv"])                                  # within the capacity: region and image stay
            assert np.array_equal(g.rtm_image_read(), before)
            if n == 1:                                                     # device signals now belong to another set
                import paper_1506_00907_b200 as pk
                with pytest.raises(pk.DGError) as e:
                    g.rtm_backward_shot(nsteps, None, updir=cfg["updir"])
                assert e.value.code == pk.DG_ERR_STATE
            data_g = g.rtm_forward_shot(nsteps)
            assert rel_l2(data_g, data_o) < TOL[precision]
            g.rtm_backward_shot(nsteps, None if n == 2 else data_o, updir=cfg["updir"])   # NULL: the recorded signals
            assert rel_l2(g.rtm_image_read(), I_sum) < (1e-10 if precision == 64 else 1e-4)
        assert g.dg_get_launch_count() > launches0
        # a receiver set beyond the capacity unbinds the region (the documented behaviour)
        import paper_1506_00907_b200 as pk
        g.dg_set_receivers(np.concatenate([cfg["receivers"], cfg["receivers"] + 0.01]))
        with pytest.raises(pk.DGError) as e:
            g.rtm_image_read()
        assert e.value.code == pk.DG_ERR_STATE
        g.close()


def test_rtm_first_image_step():
    cfg = make_config("cfg4_rtm", hexes=(4, 4, 3), N=2, nsteps=40, n_receivers_side=3)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    o = make_oracle(cfg)
    g = make_gpu(cfg, 64, history_steps=40)
    g.rtm_forward_shot(40)
    data_o, hist, qT = o.rtm_forward(40)
    # imaging over [25 dt, t_f] only == backward run of 15 steps
    g.rtm_backward_shot(40, data_o, updir=cfg["updir"], first_image_step=25)
    I_o, _, _ = o.rtm_backward(15, qT, hist, data_o, updir=cfg["updir"], nglobal_total=40)
    assert rel_l2(g.rtm_image_read(), I_o) < 1e-10
    g.close()


# ---------------------------------------------------------------------------------------------------
# config 5 shape: every order, both precisions, 3 levels
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [32, 64])
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6])
def test_cfg5_orders(N, precision):
    nsteps = 12
    cfg = make_config("cfg5_sweep", hexes=(6, 6, 8) if N < 5 else (4, 4, 5), N=N, nsteps=nsteps)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.005)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision)
    assert np.array_equal(g.dg_get_levels(), o.level)
    g.dg_step(nsteps)
    F = o.new_field()
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    assert rel_l2(g.dg_get_fields(), F.q) < TOL[precision]
    g.close()


# ---------------------------------------------------------------------------------------------------
# full BASELINE.json sizes in the launch configuration bench.py times (every CTA, every group of the
# pipelined kernel, ragged chunks): a few steps from a random state, every element compared
# ---------------------------------------------------------------------------------------------------
def per_element_max(a, b):
    """Largest per-element relative L2 error, relative to max(element norm, rms element norm): a single mis-scheduled
    block in a quiet region does not show in a global norm."""
    a, b = a.reshape(a.shape[0], -1), b.reshape(b.shape[0], -1)
    nb = np.linalg.norm(b, axis=1)
    floor = np.sqrt(np.mean(nb ** 2))
    return float((np.linalg.norm(a - b, axis=1) / np.maximum(nb, floor)).max())


@pytest.mark.parametrize("name,nsteps", [("cfg2_two_layer", 5), ("cfg4_rtm", 2), ("cfg3_lts", 1)])
def test_full_size_short_run(name, nsteps):
    """One oracle run per configuration, both precisions of the CUDA path against it (fp64: k_pipe<double,3> on configs
    2 and 4, k_step<double,4> on config 3)."""
    cfg = make_config(name)
    cfg["receivers"] = None
    o = make_oracle(cfg)
    q0 = random_state(o.K, o.Np, 11)
    F = o.new_field(q0)
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    for precision in (32, 64):
        g = make_gpu(cfg, precision)
        assert g.K == {"cfg2_two_layer": 98304, "cfg4_rtm": 786432, "cfg3_lts": 331776}[name]
        g.dg_set_state(q0)
        g.dg_step(nsteps)
        qg = g.dg_get_fields()
        assert rel_l2(qg, F.q) < TOL[precision]
        # element by element: no block of the mesh may be off
        assert per_element_max(qg, F.q) < 20 * TOL[precision]
        g.close()


@pytest.mark.parametrize("N,nsteps,levels", [(2, 4, 1), (5, 2, 1), (6, 1, 1), (4, 2, 1), (2, 1, 3)])
def test_full_size_short_run_other_orders(N, nsteps, levels):
    """The pipelined kernel at the orders it serves besides N = 3 (k_pipe<float,2 / 5 / 6>, k_pipe<double,2 / 4>; fp64 at N = 5,
    6: k_step) on the GPU-filling config-2 mesh (98 304 tetrahedra = 3 072 blocks; config-3 mesh with three levels for the
    ticket mode): a few steps from a random state against the live oracle, every element compared."""
    cfg = make_config("cfg2_two_layer" if levels == 1 else "cfg3_lts", N=N)
    cfg["receivers"] = None
    o = make_oracle(cfg)
    q0 = random_state(o.K, o.Np, 13 + N)
    F = o.new_field(q0)
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(True,))
    for precision in (32, 64):
        g = make_gpu(cfg, precision)
        assert g.K == (98304 if levels == 1 else 331776)
        g.dg_set_state(q0)
        g.dg_step(nsteps)
        qg = g.dg_get_fields()
        assert rel_l2(qg, F.q) < TOL[precision]
        assert per_element_max(qg, F.q) < 20 * TOL[precision]
        g.close()


@pytest.mark.parametrize("name", ["cfg2_two_layer", "cfg3_lts", "cfg4_rtm"])
def test_full_size_full_length_fp32_against_fp64(name):
    """BASELINE.json configs 2, 3, 4 at FULL size and FULL length (1000 steps; 500 global steps of three levels at N = 4; 2000
    steps), in the launch configuration bench.py times: the oracle cannot run these, so the fp32 path is compared with the
    fp64 path of the library, which is itself pinned to the oracle at full length on the 41 472-element meshes
    (tests/test_gpu_goldens.py) and at full size over a few steps (test_full_size_short_run).  north_star: relative L2
    <= 1e-5 in fp32 after the stated step counts."""
    cfg = make_config(name)
    cfg["receivers"] = None
    q = {}
    for precision in (64, 32):
        g = make_gpu(cfg, precision)
        g.dg_step(cfg["nsteps"])
        q[precision] = g.dg_get_fields()
        g.close()
    assert np.linalg.norm(q[64]) > 0
    err = rel_l2(q[32], q[64])
    assert err < TOL[32], err
    assert per_element_max(q[32], q[64]) < 20 * TOL[32]


def test_full_size_rtm_two_steps():
    """Config 4 at full size (786 432 tetrahedra, 32 768 stored boundary faces): two forward steps with trace capture and
    receiver recording, two backward steps of both wavefields with replay, injection and imaging, against the live
    oracle.  A 16 x 16 receiver grid plus receivers around the source (the oracle locates receivers by brute force; the
    64 x 64 grid is covered at full length by tests/test_gpu_goldens.py); from rest the fields are non-zero only near the
    source and the receivers after two steps, so this checks the indexing at full size (every stored face, every
    block: zeros must stay zeros) rather than the arithmetic."""
    nsteps = 2
    cfg = make_config("cfg4_rtm", n_receivers_side=16)
    x0 = cfg["source"]["x0"]
    h = cfg["lengths"][0] / cfg["hexes"][0]
    ring = x0[None, :] + h * np.array([[0.02, 0.03, 0.01], [0.21, -0.13, 0.05], [-0.17, 0.22, -0.04], [0.35, 0.31, 0.12],
                                       [-0.4, -0.28, 0.2], [0.05, -0.45, 0.3]])
    cfg["receivers"] = np.concatenate([cfg["receivers"], ring])
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.002)
    o = make_oracle(cfg)
    data_o, hist, qT = o.rtm_forward(nsteps)
    assert np.abs(data_o).max() > 0
    d = 0.5 * data_o + 1e-3 * np.abs(data_o).max() * np.random.default_rng(3).standard_normal(data_o.shape)
    I_o, FS, FR = o.rtm_backward(nsteps, qT, hist, d, updir=cfg["updir"], nglobal_total=nsteps)
    assert np.abs(I_o).max() > 0
    for precision in (32, 64):
        tol = TOL[precision]
        g = make_gpu(cfg, precision, history_steps=nsteps)
        data_g = g.rtm_forward_shot(nsteps)
        assert rel_l2(data_g, data_o) < tol
        faces, nrec = g.rtm_get_trace_index(0)
        assert faces.size == 32768 and np.array_equal(faces, hist.faces[0]) and nrec == nsteps + 1
        for j in range(nrec):
            assert np.abs(g.rtm_get_traces(0, j) - hist.records[0][j]).max() <= 10 * tol * np.abs(hist.records[0]).max()
        assert rel_l2(g.rtm_get_fields(0), qT) < tol
        g.rtm_backward_shot(nsteps, d, updir=cfg["updir"])
        assert rel_l2(g.rtm_get_fields(1), FS.q) < 3 * tol
        assert rel_l2(g.rtm_get_fields(2), FR.q) < 3 * tol
        assert per_element_max(g.rtm_get_fields(2), FR.q) < 60 * tol
        I_g = g.rtm_image_read()
        assert rel_l2(I_g, I_o) < (1e-4 if precision == 32 else 1e-10)
        assert per_element_max(I_g, I_o) < (1e-3 if precision == 32 else 1e-9)
        g.close()


@pytest.mark.parametrize("N", [3, 4])
def test_tensor_core_variant_is_close_but_opt_in(N, monkeypatch):
    """The tcgen05 / tensor-memory variant of the step kernel (DGRTM_KERNEL=tc, fp32, N = 3 and 4, 3xTF32 split) is NOT
    the default: it does not hold the 1e-5 fp32 tolerance over a 1000-step run (1.4e-5 measured on config 2) and is not
    faster (N = 4: one group per SM, the split A operand fills the tensor memory).  It must still be a
    correct implementation of the same step to TF32x3 accuracy."""
    cfg = make_config("cfg2_two_layer", hexes=(6, 5, 4), N=N, nsteps=200)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.005)
    o = make_oracle(cfg)
    monkeypatch.setenv("DGRTM_KERNEL", "tc")
    g = make_gpu(cfg, 32)
    monkeypatch.delenv("DGRTM_KERNEL")
    g.dg_step(200)
    F = o.new_field()
    o.run_mrab([F], 200, 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    err = rel_l2(g.dg_get_fields(), F.q)
    assert err < 1e-4, err
    g.close()


# ---------------------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------------------
def test_single_element_and_tiny_meshes():
    """K = 1 (all four faces on the boundary, one lane of one block) and K = 6."""
    for etov, vx in ((np.array([[0, 1, 2, 3]], dtype=np.int32),
                      np.array([[0.0, 0, 0], [1.0, 0, 0], [0, 1.0, 0], [0, 0, 1.0]])),
                     box_tet_mesh(1, 1, 1)):
        K = etov.shape[0]
        cfg = dict(EToV=etov, VX=vx, rho=np.full(K, 1.3), c=np.full(K, 2.0), N=3, precision=64, default_bc=2,
                   nlevels=1, cfl=0.15, source=None, receivers=None)
        o = make_oracle(cfg)
        g = make_gpu(cfg, 64)
        q0 = random_state(K, o.Np, 3)
        g.dg_set_state(q0)
        F = o.new_field(q0)
        g.dg_step(20)
        o.run_mrab([F], 20, 0.0, 1, source_on=(False,))
        assert rel_l2(g.dg_get_fields(), F.q) < TOL[64]
        g.close()


def test_error_paths():
    import paper_1506_00907_b200 as pk
    etov, vx = box_tet_mesh(2, 2, 2)
    bad = etov.copy()
    bad[3, [0, 1]] = bad[3, [1, 0]]                       # negatively oriented tet
    with pytest.raises(pk.DGError) as e:
        pk.DG(2, 64, bad, vx)
    assert e.value.code == pk.DG_ERR_MESH and "3" in str(e.value)
    with pytest.raises(pk.DGError) as e:
        pk.DG(7, 64, etov, vx)
    assert e.value.code == pk.DG_ERR_UNSUPPORTED
    with pytest.raises(pk.DGError) as e:
        pk.DG(2, 16, etov, vx)
    assert e.value.code == pk.DG_ERR_UNSUPPORTED
    g = pk.DG(2, 64, etov, vx)
    with pytest.raises(pk.DGError) as e:
        g.dg_workspace_bytes()
    assert e.value.code == pk.DG_ERR_STATE
    K = etov.shape[0]
    with pytest.raises(pk.DGError) as e:
        g.dg_set_model(np.ones(K), -np.ones(K))
    assert e.value.code == pk.DG_ERR_ARG
    g.dg_set_model(np.ones(K), np.ones(K))
    with pytest.raises(pk.DGError) as e:
        g.dg_step(1)
    assert e.value.code == pk.DG_ERR_STATE
    with pytest.raises(pk.DGError) as e:
        g.dg_set_source([5.0, 5.0, 5.0], 10.0, 0.1)
    assert e.value.code == pk.DG_ERR_ARG
    import torch
    n = g.dg_workspace_bytes()
    buf = torch.empty(n + 256, dtype=torch.uint8, device="cuda:0")
    base = (buf.data_ptr() + 255) & ~255
    with pytest.raises(pk.DGError) as e:
        g.dg_bind_workspace(base, n - 1)
    assert e.value.code == pk.DG_ERR_NOMEM
    with pytest.raises(pk.DGError) as e:
        g.dg_bind_workspace(base + 8, n)
    assert e.value.code == pk.DG_ERR_ARG
    g.dg_bind_workspace(base, n, torch.cuda.current_stream().cuda_stream)
    with pytest.raises(pk.DGError) as e:
        g.rtm_forward_shot(3, want_data=False)
    assert e.value.code == pk.DG_ERR_STATE
    g.dg_step(0)
    g.close()


def test_shuffled_element_order_gives_the_same_fields():
    """The user's element order never shows in the result (the library un-permutes)."""
    etov, vx = box_tet_mesh(3, 3, 3, jitter=0.1, seed=5)
    etov2, perm = permute_elements(etov, 6)
    K = etov.shape[0]
    base = dict(VX=vx, N=3, precision=64, default_bc=2, nlevels=1, cfl=0.15, source=None, receivers=None)
    rng = np.random.default_rng(1)
    rho, c = rng.uniform(1, 2, K), rng.uniform(1.5, 3, K)
    cfgA = dict(base, EToV=etov, rho=rho, c=c)
    cfgB = dict(base, EToV=etov2, rho=rho[perm], c=c[perm])
    gA, gB = make_gpu(cfgA, 64), make_gpu(cfgB, 64)
    q0 = random_state(K, gA.Np, 9)
    gA.dg_set_state(q0)
    gB.dg_set_state(q0[perm])
    gA.dg_step(10)
    gB.dg_step(10)
    assert rel_l2(gB.dg_get_fields(), gA.dg_get_fields()[perm]) < 1e-12
    gA.close()
    gB.close()
