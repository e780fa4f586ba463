"""Every boundary type and oblique / horizontal characteristic directions STEPPED through the fused kernels (k_pipe,
k_step) against the oracle - SURVEY.md 8(f) item 1:

  * free surface p = 0 and transparent boundary, eq (3); rigid wall (config 1) and prescribed exterior
    (plane-wave pin), reading Q6; the stand-alone k_rhs sees them in test_gpu_parity.py::test_rhs_volume_surface, here
    the kernels that actually advance the fields do, forward and backward (tau < 0);
  * an RTM shot with a free-surface top, a rigid bottom and absorbing sides (only absorbing faces are stored, Q12);
  * imaging along e_z, an oblique direction and e_x.
"""
import numpy as np
import pytest

from workloads import box_tet_mesh, box_side_bc, make_config, permute_elements
from parity_util import make_oracle, make_gpu, rel_l2, random_state

pytestmark = pytest.mark.gpu

TOL = {64: 1e-10, 32: 1e-5}


def per_element_max(a, b):
    """Largest per-element relative L2 error, relative to max(element norm, rms element norm)."""
    a, b = a.reshape(a.shape[0], -1), b.reshape(b.shape[0], -1)
    nb = np.linalg.norm(b, axis=1)
    floor = np.sqrt(np.mean(nb ** 2))
    return float((np.linalg.norm(a - b, axis=1) / np.maximum(nb, floor)).max())


def mixed_bc_cfg(N, hexes=(4, 4, 3), seed=21):
    """Jittered box, shuffled element order, all four boundary types (by centroid quadrant), random material."""
    etov, vx = box_tet_mesh(*hexes, lengths=(1.5, 1.5, 1.0), jitter=0.1, seed=seed)
    etov, _ = permute_elements(etov, seed + 1)
    K = etov.shape[0]
    rng = np.random.default_rng(seed)
    cen = vx[etov].mean(axis=1)
    face_bc = np.zeros((K, 4), dtype=np.int8)
    face_bc[:] = (1 + (cen[:, 0] > 0.75).astype(int) + 2 * (cen[:, 1] > 0.75).astype(int))[:, None]
    cfg = dict(EToV=etov, VX=vx, rho=rng.uniform(1.0, 2.5, K), c=rng.uniform(1.5, 4.5, K), N=N, precision=64,
               default_bc=2, nlevels=1, cfl=0.15, source=None, receivers=None)
    return cfg, face_bc


@pytest.mark.parametrize("N,precision,kernel", [(3, 32, "pipe"), (4, 32, "pipe"), (3, 64, "pipe"), (3, 32, "step"),
                                                (2, 64, "step"), (5, 64, "step"), (1, 32, "step"), (6, 32, "step"),
                                                (4, 64, "step")])
def test_all_boundary_types_stepped(N, precision, kernel, monkeypatch):
    cfg, face_bc = mixed_bc_cfg(N)
    o = make_oracle(cfg, face_bc=face_bc)
    assert set(np.unique(o.bc[o.bnd_k, o.bnd_f])) == {1, 2, 3, 4}
    if kernel == "step":
        monkeypatch.setenv("DGRTM_KERNEL", "step")
    g = make_gpu(cfg, precision, face_bc=face_bc)
    monkeypatch.delenv("DGRTM_KERNEL", raising=False)
    nsteps = 200
    q0 = random_state(o.K, o.Np, 300 + N)
    ext = np.random.default_rng(9).standard_normal((o.bnd_k.size, o.Nfp, 2))
    presc = o.bc[o.bnd_k, o.bnd_f] == 4
    ext_o = np.where(presc[:, None, None], ext, 0.0)        # the oracle applies `exterior` to absorbing faces too
    g.dg_set_state(q0)
    g.dg_set_exterior(ext)
    g.dg_step(nsteps)
    F = o.new_field(q0)
    o.run_mrab([F], nsteps, 0.0, 1, source_on=(False,), exterior_fn=lambda t: ext_o)
    qg = g.dg_get_fields()
    assert rel_l2(qg, F.q) < TOL[precision], rel_l2(qg, F.q)
    assert per_element_max(qg, F.q) < 10 * TOL[precision]
    assert rel_l2(g.dg_get_traces(), F.qf) < TOL[precision]
    g.close()


@pytest.mark.parametrize("N,precision", [(3, 64), (2, 64), (3, 32), (4, 32)])
def test_plane_wave_with_prescribed_exterior_refreshed_every_step(N, precision):
    """p = g(k.x - ct), v = k g/(rho c) with the exterior traces prescribed from the exact solution at every step
    start (dg_set_exterior before each dg_step(1)) - the plane-wave pin of SURVEY.md 8(c) through the stepping kernel."""
    rho, c = 1.3, 2.0
    khat = np.array([2.0, 1.0, -2.0]) / 3.0
    gfun = lambda s: np.exp(-(s / 0.25) ** 2)
    etov, vx = box_tet_mesh(4, 4, 4, jitter=0.1, seed=5)
    K = etov.shape[0]
    cfg = dict(EToV=etov, VX=vx, rho=np.full(K, rho), c=np.full(K, c), N=N, precision=precision, default_bc=4,
               nlevels=1, cfl=0.15, source=None, receivers=None)
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision)

    def exact(t):
        s = o.X @ khat - 0.5 - c * t
        q = np.zeros((K, 4, o.Np))
        q[:, 0] = gfun(s)
        for i in range(3):
            q[:, 1 + i] = khat[i] * gfun(s) / (rho * c)
        return q

    def exterior(t):
        return o.traces_of(exact(t), np.arange(K))[o.bnd_k, o.bnd_f]

    nsteps = 40
    g.dg_set_state(exact(0.0))
    for n in range(nsteps):
        g.dg_set_exterior(exterior(n * o.dt_local))
        if n % 2:
            g.dg_halo_sources([])                                 # fused exchange switched on with no halo face: every
        g.dg_step(1)                                              # prescribed face must still read the exterior array
    F = o.new_field(exact(0.0))
    t_end = o.run_mrab([F], nsteps, 0.0, 1, source_on=(False,), exterior_fn=exterior)
    qg = g.dg_get_fields()
    assert rel_l2(qg, F.q) < TOL[precision]
    assert per_element_max(qg, F.q) < 10 * TOL[precision]
    assert rel_l2(qg, exact(t_end)) < 0.05                        # discretisation error only
    g.close()


def _shot_cfg(N, nsteps, hexes=(5, 4, 3)):
    cfg = make_config("cfg4_rtm", hexes=hexes, N=N, nsteps=nsteps, n_receivers_side=3)
    cfg["source"] = dict(cfg["source"], f0=60.0, tp=0.01)
    return cfg


@pytest.mark.parametrize("N,precision", [(3, 32), (3, 64), (2, 64), (4, 32), (5, 32)])
def test_rtm_shot_with_free_surface_top(N, precision):
    """Free-surface top (eq (3) neighbour p = 0), rigid bottom, absorbing sides: the mirror conditions are
    time-reversible and are not stored; the absorbing sides are captured and replayed (reading Q12)."""
    nsteps = 60
    cfg = _shot_cfg(N, nsteps)
    face_bc = box_side_bc(cfg["EToV"], cfg["VX"], cfg["lengths"], top=1, bottom=3, sides=2)
    o = make_oracle(cfg, face_bc=face_bc)
    kinds = o.bc[o.bnd_k, o.bnd_f]
    assert (kinds == 1).sum() > 0 and (kinds == 3).sum() > 0 and (kinds == 2).sum() > 0
    g = make_gpu(cfg, precision, face_bc=face_bc, history_steps=nsteps)
    tol = TOL[precision]
    data_g = g.rtm_forward_shot(nsteps)
    data_o, hist, qT = o.rtm_forward(nsteps)
    assert np.abs(data_o).max() > 0
    faces, nrec = g.rtm_get_trace_index(0)
    assert np.array_equal(faces, hist.faces[0]) and faces.size == (kinds == 2).sum()
    assert rel_l2(data_g, data_o) < tol
    assert rel_l2(g.rtm_get_fields(0), qT) < tol
    assert per_element_max(g.rtm_get_fields(0), qT) < 10 * tol
    g.rtm_backward_shot(nsteps, data_o, updir=cfg["updir"])
    I_o, FS, FR = o.rtm_backward(nsteps, qT, hist, data_o, updir=cfg["updir"], nglobal_total=nsteps)
    assert rel_l2(g.rtm_get_fields(1), FS.q) < 3 * tol
    assert rel_l2(g.rtm_get_fields(2), FR.q) < 3 * tol
    assert np.abs(I_o).max() > 0
    assert rel_l2(g.rtm_image_read(), I_o) < (1e-4 if precision == 32 else 1e-10)
    g.close()


@pytest.mark.parametrize("updir", [(0.3, -0.2, -0.93), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)])
@pytest.mark.parametrize("N,precision", [(3, 32), (2, 64), (4, 32)])
def test_rtm_shot_oblique_and_horizontal_directions(N, precision, updir):
    """Characteristic imaging (7)-(8) along an oblique unit vector, e_x, e_y and +e_z: a swapped or
    dropped component of the direction would pass every test that images along (0, 0, -1)."""
    e = np.asarray(updir, dtype=np.float64)
    e = e / np.linalg.norm(e)
    nsteps = 40
    cfg = _shot_cfg(N, nsteps, hexes=(4, 4, 3))
    o = make_oracle(cfg)
    g = make_gpu(cfg, precision, history_steps=nsteps)
    g.rtm_forward_shot(nsteps, want_data=False)
    data_o, hist, qT = o.rtm_forward(nsteps)
    g.rtm_backward_shot(nsteps, data_o, updir=e)
    I_o, _, _ = o.rtm_backward(nsteps, qT, hist, data_o, updir=e, nglobal_total=nsteps)
    I_z, _, _ = o.rtm_backward(nsteps, qT, hist, data_o, updir=(0.0, 0.0, -1.0), nglobal_total=nsteps)
    assert np.abs(I_o).max() > 0 and rel_l2(I_o, I_z) > 1e-3           # the direction matters
    I_g = g.rtm_image_read()
    assert rel_l2(I_g, I_o) < (1e-4 if precision == 32 else 1e-10)
    assert per_element_max(I_g, I_o) < (1e-3 if precision == 32 else 1e-9)
    g.close()
