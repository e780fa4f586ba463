"""Pins for the oracle's DG scheme as a whole (CPU only): what the paper and the mathematics fix.

  * right-hand side of a globally linear field is exact (jumps vanish);
  * discrete energy-rate identity of the penalty fluxes (11)-(12), face integrals evaluated
    independently by quadrature at physical points, both time directions;
  * closed-form rigid-cavity mode and plane wave, h^{N+1} rates;
  * third-order convergence in dt of the AB3 update (18);
  * multi-rate run (Algorithm 1) vs single-rate run at dt_local; level assignment by brute force;
  * point-source weights (15); imaging accumulation properties; trace replay reconstruction.
"""
import numpy as np
import pytest

from oracle.dgtd import (DGOracle, assign_levels, ricker, BC_ABSORBING, BC_RIGID, BC_FREE,
                         BC_PRESCRIBED)
from oracle.reference_element import tri_quadrature
from oracle.coefficients import ab_coefficients
from workloads import box_tet_mesh, graded_box_tet_mesh, make_config


def cavity_exact(X, t, rho=1.0, c=1.0):
    w = np.sqrt(3.0) * np.pi * c
    cx, cy, cz = [np.cos(np.pi * X[..., d]) for d in range(3)]
    sx, sy, sz = [np.sin(np.pi * X[..., d]) for d in range(3)]
    q = np.zeros(X.shape[:2][:1] + (4,) + X.shape[1:2])
    q[:, 0] = cx * cy * cz * np.cos(w * t)
    a = np.pi / (rho * w) * np.sin(w * t)
    q[:, 1] = a * sx * cy * cz
    q[:, 2] = a * cx * sy * cz
    q[:, 3] = a * cx * cy * sz
    return q


def test_rhs_of_linear_field_is_exact():
    etov, vx = box_tet_mesh(2, 2, 2, jitter=0.1, seed=11)
    dg = DGOracle(2, etov, vx, default_bc=BC_PRESCRIBED)
    K = dg.K
    dg.set_model(np.full(K, 1.7), np.full(K, 2.3))
    X = dg.X
    a = np.array([0.3, -0.7, 0.5])
    B = np.array([[0.2, 0.1, -0.3], [0.0, -0.4, 0.6], [0.5, 0.2, 0.1]])
    q = np.zeros((K, 4, dg.Np))
    q[:, 0] = 1.0 + X @ a
    for i in range(3):
        q[:, 1 + i] = 0.1 * i + X @ B[i]
    F = dg.new_field(q)
    # prescribed exterior = the same linear field -> all jumps vanish
    ext = F.qf[dg.bnd_k, dg.bnd_f].copy()
    r = dg.rhs(F.q, F.qf, 0.0, exterior=ext, source_on=False)
    assert np.abs(r[:, 0] - (-1.7 * 2.3 ** 2 * np.trace(B))).max() < 1e-11
    for i in range(3):
        assert np.abs(r[:, 1 + i] - (-a[i] / 1.7)).max() < 1e-11
    assert np.abs(dg.rhs_surface(F.q, F.qf, exterior=ext)).max() < 1e-11


def _face_points(f, u, v):
    m1 = -np.ones_like(u)
    return [(u, v, m1), (u, m1, v), (-1 - u - v, u, v), (m1, u, v)][f]


@pytest.mark.parametrize("direction", [1, -1])
def test_energy_rate_identity(direction):
    etov, vx = box_tet_mesh(2, 2, 1, jitter=0.15, seed=21)
    rng = np.random.default_rng(3)
    K = etov.shape[0]
    face_bc = rng.integers(1, 4, size=(K, 4)).astype(np.int8)      # free / absorbing / rigid mix
    dg = DGOracle(3, etov, vx, face_bc=face_bc)
    dg.set_model(rng.uniform(1.0, 2.5, K), rng.uniform(1.5, 4.5, K))
    q = rng.standard_normal((K, 4, dg.Np))
    F = dg.new_field(q)
    r = dg.rhs(F.q, F.qf, 0.0, direction=direction, source_on=False)
    M, J = dg.ref.M, dg.geo["J"]
    lhs = 0.0
    for k in range(K):
        lhs += J[k] * (q[k, 0] @ M @ r[k, 0] / (dg.rho[k] * dg.c[k] ** 2)
                       + dg.rho[k] * sum(q[k, 1 + i] @ M @ r[k, 1 + i] for i in range(3)))
    # right-hand side of the identity by quadrature at physical points (independent of LIFT/mapP)
    u, v, w = tri_quadrature(dg.N + 2)
    rhs_val = 0.0

    def values_at(k, x_phys):
        v0 = dg.VX[dg.EToV[k, 0]]
        rst = np.einsum("ij,ni->nj", dg.geo["ginv"][k], x_phys - v0) - 1.0
        rows = np.array([dg.ref.interp_row(*p) for p in rst])
        return rows @ q[k].T                                       # [nq,4]

    for k in range(K):
        for f in range(4):
            rr, ss, tt = _face_points(f, u, v)
            lam = np.stack([-(1 + rr + ss + tt) / 2, (1 + rr) / 2, (1 + ss) / 2, (1 + tt) / 2], axis=1)
            xq = lam @ dg.VX[dg.EToV[k]]
            wq = w * dg.geo["area"][k, f] / 2.0
            n = dg.geo["normals"][k, f]
            own = values_at(k, xq)
            pm, nvm = own[:, 0], own[:, 1:4] @ n
            k2 = dg.EToE[k, f]
            if k2 >= 0:
                if k2 < k:
                    continue                                       # interior faces once
                oth = values_at(k2, xq)
                dp, dnv = oth[:, 0] - pm, oth[:, 1:4] @ n - nvm
                Zf = 0.5 * (dg.Z[k] + dg.Z[k2])
                rhs_val -= np.sum(wq * 0.5 * (direction / Zf * dp ** 2 + direction * Zf * dnv ** 2))
            else:
                Z = dg.Z[k]
                tp, tv = direction / Z, direction * Z
                if dg.bc[k, f] == BC_ABSORBING:
                    rhs_val -= np.sum(wq * 0.5 * (tp * pm ** 2 + tv * nvm ** 2))
                elif dg.bc[k, f] == BC_RIGID:
                    rhs_val -= np.sum(wq * tv * nvm ** 2)
                elif dg.bc[k, f] == BC_FREE:
                    rhs_val -= np.sum(wq * tp * pm ** 2)
    assert abs(lhs - rhs_val) < 1e-10 * max(1.0, abs(rhs_val))
    assert (rhs_val < 0) if direction == 1 else (rhs_val > 0)


@pytest.mark.parametrize("N", [2, 3])
def test_cavity_mode_convergence_lserk4(N):
    errs = []
    for n in (2, 4):
        cfg = make_config("cfg1_cavity", hexes=(n, n, n), N=N)
        dg = DGOracle(N, cfg["EToV"], cfg["VX"], default_bc=BC_RIGID)
        dg.set_model(cfg["rho"], cfg["c"], 1, 0.5)
        F = dg.new_field(cavity_exact(dg.X, 0.0))
        T = 0.3
        ns = int(np.ceil(T / dg.dt_local))
        t = dg.run_lserk4(F, 0.0, T / ns, ns)
        e = cavity_exact(dg.X, t)
        errs.append(np.linalg.norm(F.q - e) / np.linalg.norm(e))
    rate = np.log2(errs[0] / errs[1])
    assert rate > N + 0.4, (errs, rate)          # h^{N+1}
    assert errs[1] < 0.05


def test_plane_wave_with_prescribed_exterior():
    """p = g(k.x - ct), v = k g/(rho c) is an exact solution; exterior states prescribed."""
    rho, c = 1.3, 2.0
    khat = np.array([2.0, 1.0, -2.0]) / 3.0
    g = lambda s: np.exp(-(s / 0.25) ** 2)
    errs = []
    for n in (2, 4):
        etov, vx = box_tet_mesh(n, n, n, jitter=0.1, seed=5)
        dg = DGOracle(3, etov, vx, default_bc=BC_PRESCRIBED)
        dg.set_model(np.full(dg.K, rho), np.full(dg.K, c), 1, 0.5)

        def exact(t, X=dg.X):
            s = X @ khat - 0.5 - c * t
            q = np.zeros((dg.K, 4, dg.Np))
            q[:, 0] = g(s)
            for i in range(3):
                q[:, 1 + i] = khat[i] * g(s) / (rho * c)
            return q

        def exterior(t):
            qf = dg.traces_of(exact(t), np.arange(dg.K))
            return qf[dg.bnd_k, dg.bnd_f]

        F = dg.new_field(exact(0.0))
        T = 0.1
        ns = int(np.ceil(T / dg.dt_local))
        t = dg.run_lserk4(F, 0.0, T / ns, ns, exterior_fn=exterior)
        e = exact(t)
        errs.append(np.linalg.norm(F.q - e) / np.linalg.norm(e))
    assert errs[1] < 0.02 and np.log2(errs[0] / errs[1]) > 3.0, errs


def test_ab3_third_order_in_time_and_energy_decay():
    cfg = make_config("cfg1_cavity", hexes=(2, 2, 2), N=3)
    dg = DGOracle(3, cfg["EToV"], cfg["VX"], default_bc=BC_RIGID)
    K = dg.K
    # semi-discrete reference: LSERK4 with a tiny step
    dg.set_model(cfg["rho"], cfg["c"], 1, 0.02)
    q0 = cavity_exact(dg.X, 0.0)
    T = 0.2
    F = dg.new_field(q0)
    ns = int(np.ceil(T / dg.dt_local))
    dg.run_lserk4(F, 0.0, T / ns, ns)
    qref = F.q.copy()
    errs = []
    for nsteps in (40, 80):
        dt = T / nsteps
        dg.dt_local = dt
        dg.dt_global = dt
        # exact-history priming: rhs at -dt, -2dt from a backward LSERK4 run of the semi-discrete
        # system (so the start-up ramp, reading Q7, does not limit the order)
        F = dg.new_field(q0)
        G = dg.new_field(q0)
        hist = []
        for j in (1, 2):
            dg.run_lserk4(G, 0.0, -dt / 8, 8)
            hist.append(dg.rhs(G.q, G.qf, 0.0, source_on=False))
        F.hist[0], F.hist[1] = hist[0], hist[1]       # become slots 1, 2 after the first evaluation
        F.nhist[:] = 2
        dg.run_mrab([F], nsteps, 0.0, 1, source_on=(False,))
        errs.append(np.linalg.norm(F.q - qref) / np.linalg.norm(qref))
    assert np.log2(errs[0] / errs[1]) > 2.7, errs
    # discrete energy does not grow over an AB3 run with absorbing walls
    dg2 = DGOracle(2, cfg["EToV"], cfg["VX"], default_bc=BC_ABSORBING)
    dg2.set_model(cfg["rho"], cfg["c"], 1, 0.15)
    F = dg2.new_field(cavity_exact(dg2.X, 0.0))

    def energy(q):
        e = 0.0
        for fld in range(4):
            e += np.einsum("k,kn,nm,km->", dg2.geo["J"], q[:, fld], dg2.ref.M, q[:, fld])
        return 0.5 * e
    E = [energy(F.q)]
    for _ in range(10):
        dg2.run_mrab([F], 5, 0.0, 1, source_on=(False,))
        E.append(energy(F.q))
    assert np.all(np.diff(E) < 1e-12) and E[-1] < 0.9 * E[0]


def _lts_setup(N=2, nlevels=3, cfl=0.15):
    etov, vx = graded_box_tet_mesh(4, 4, 8, (1.0, 1.0, 1.0), band_center=0.5, band_width=0.2,
                                   max_ratio=4.0, seed=9, blob_sigma_cells=1.0)
    dg = DGOracle(N, etov, vx, default_bc=BC_ABSORBING)
    zc = vx[etov].mean(axis=1)[:, 2]
    c = np.where((zc > 0.8) | (zc < 0.2), 1.0, 2.0)
    dg.set_model(np.ones(dg.K), c, nlevels, cfl)
    return dg


def test_level_assignment_bruteforce():
    dg = _lts_setup()
    L = dg.nlevels
    K = dg.K
    assert len(np.unique(dg.level)) == 3, np.bincount(dg.level)
    raw = np.zeros(K, dtype=int)
    for k in range(K):
        j = 0
        while j + 1 <= L - 1 and 2.0 ** (j + 1) * dg.dt_local <= dg.dt_k[k]:
            j += 1
        raw[k] = j
    # graph distance by BFS from every element; j_k = min_m raw_m + d(k,m)  (reading Q9)
    nbrs = [[int(x) for x in dg.EToE[k] if x >= 0] for k in range(K)]
    best = raw.copy()
    for src in range(K):
        dist = {src: 0}
        frontier = [src]
        while frontier and max(dist.values()) < L:
            nxt = []
            for a in frontier:
                for b in nbrs[a]:
                    if b not in dist:
                        dist[b] = dist[a] + 1
                        nxt.append(b)
            frontier = nxt
        for k, d in dist.items():
            best[k] = min(best[k], raw[src] + d)
    assert np.array_equal(dg.level, (L - 1) - best)
    # invariants: neighbours differ by at most one level; never coarser than raw
    for k in range(K):
        for b in nbrs[k]:
            assert abs(int(dg.level[k]) - int(dg.level[b])) <= 1
    assert np.all((L - 1) - dg.level <= raw)
    assert np.all(2.0 ** ((L - 1) - dg.level) * dg.dt_local <= dg.dt_k * (1 + 1e-14))


def test_multirate_agrees_with_single_rate():
    """Algorithm 1 with 3 levels vs the single-rate scheme at dt_local: same semi-discrete system,
    both third order -> the difference is O(dt^3) and small; refining dt by 2 cuts it by ~8."""
    diffs = []
    for cfl in (0.15, 0.075):
        dg = _lts_setup(cfl=cfl)
        x0 = np.array([0.52, 0.47, 0.31])
        dg.set_source(x0, f0=5.0, tp=0.2, amp=1.0)
        T_glob = int(round(0.3 / dg.dt_global))
        F = dg.new_field()
        dg.run_mrab([F], T_glob, 0.0, 1)
        lev, dtl = dg.level.copy(), dg.dt_local
        # single rate: all elements on the finest level, same dt_local
        dg.nlevels, dg.level = 1, np.zeros(dg.K, dtype=np.int32)
        dg.nlocal, dg.dt_global = 1, dtl
        dg.has_finer_nbr[:] = False
        G = dg.new_field()
        dg.run_mrab([G], T_glob * 4, 0.0, 1)
        diffs.append(np.linalg.norm(F.q - G.q) / np.linalg.norm(G.q))
    assert diffs[0] < 5e-3, diffs
    assert diffs[0] / diffs[1] > 4.0, diffs


def test_point_source_weights():
    etov, vx = box_tet_mesh(2, 2, 2, jitter=0.1, seed=13)
    dg = DGOracle(3, etov, vx)
    dg.set_model(np.ones(dg.K), np.ones(dg.K))
    x0 = np.array([0.61, 0.33, 0.42])
    k, ell, w = dg.point_weights(x0)
    Mk = dg.geo["J"][k] * dg.ref.M
    assert abs(np.sum(Mk @ w) - 1.0) < 1e-12               # int delta~ = 1
    assert abs(ell.sum() - 1.0) < 1e-12
    X = dg.X[k]
    for (a, b, c) in [(1, 0, 0), (0, 2, 0), (1, 1, 1), (0, 0, 3)]:
        gfun = lambda x: x[..., 0] ** a * x[..., 1] ** b * x[..., 2] ** c
        assert abs(gfun(X) @ Mk @ w - gfun(x0)) < 1e-11     # (g, delta~) = g(x0), deg <= N
        assert abs(ell @ gfun(X) - gfun(x0)) < 1e-11
    # the point is inside the located element
    lam = np.linalg.solve(np.vstack([dg.VX[dg.EToV[k]].T, np.ones(4)]), np.append(x0, 1.0))
    assert lam.min() > -1e-12
    assert abs(ricker(0.1, 15.0, 0.1) - 1.0) < 1e-15 and abs(ricker(0.0, 15.0, 0.1)) < 1e-7


def _small_rtm(nglobal=30, nlevels=1):
    etov, vx = box_tet_mesh(3, 3, 2, lengths=(1.5, 1.5, 1.0), jitter=0.1, seed=17)
    dg = DGOracle(2, etov, vx, default_bc=BC_ABSORBING)
    c = np.where(vx[etov].mean(axis=1)[:, 2] > 0.6, 2.2, 1.5)
    dg.set_model(np.ones(dg.K), c, nlevels, 0.15)
    dg.set_source(np.array([0.77, 0.74, 0.13]), f0=8.0, tp=0.02, amp=1.0)
    gx = np.linspace(0.2, 1.3, 3)
    xr = np.array([[x + 0.003, y + 0.007, 0.11] for x in gx for y in gx])
    dg.set_receivers(xr)
    return dg


def test_trace_replay_reconstructs_the_forward_field():
    """Backward run with negative penalties and replayed boundary traces
    returns to the initial state at discretisation level (soft pin, reading Q12): the error falls
    with N and is far below that of a backward run without replay."""
    from oracle.dgtd import TraceHistory
    etov, vx = box_tet_mesh(3, 3, 2, lengths=(1.5, 1.5, 1.0), jitter=0.1, seed=17)
    rel = {}
    for N in (2, 4):
        dg = DGOracle(N, etov, vx, default_bc=BC_ABSORBING)
        dg.set_model(np.ones(dg.K), np.full(dg.K, 1.5), 1, 0.15)
        q0 = np.zeros((dg.K, 4, dg.Np))
        q0[:, 0] = np.exp(-np.sum((dg.X - np.array([0.75, 0.75, 0.4])) ** 2, axis=2) / 0.3 ** 2)
        ng = int(0.5 / dg.dt_global)
        F = dg.new_field(q0)
        hist = TraceHistory(dg, ng)
        dg.run_mrab([F], ng, 0.0, 1, source_on=(False,), capture=hist, first_fine_index=0)
        assert np.linalg.norm(F.q) < 0.7 * np.linalg.norm(q0)        # part of the pulse has left
        FS = dg.new_field(F.q)
        dg.run_mrab([FS], ng, ng * dg.dt_global, -1, source_on=(False,), replay=hist,
                    first_fine_index=ng)
        rel[N] = np.linalg.norm(FS.q - q0) / np.linalg.norm(q0)
        if N == 2:
            FN = dg.new_field(F.q)
            dg.run_mrab([FN], ng, ng * dg.dt_global, -1, source_on=(False,), first_fine_index=ng)
            assert rel[N] < 0.5 * np.linalg.norm(FN.q - q0) / np.linalg.norm(q0)
    assert rel[4] < 0.08 and rel[4] < 0.4 * rel[2], rel


def test_image_accumulation_properties():
    dg = _small_rtm()
    nglobal = 40
    data, hist, qT = dg.rtm_forward(nglobal)
    assert np.abs(data).max() > 0
    I, FS, FR = dg.rtm_backward(nglobal // 2, qT, hist, data, nglobal_total=nglobal)
    assert np.abs(I).max() > 0
    # zero data -> zero image; bilinearity in the data
    I0, _, _ = dg.rtm_backward(nglobal // 2, qT, hist, 0 * data, nglobal_total=nglobal)
    assert np.abs(I0).max() == 0.0
    I2, _, _ = dg.rtm_backward(nglobal // 2, qT, hist, -2.5 * data, nglobal_total=nglobal)
    assert np.allclose(I2, -2.5 * I, rtol=1e-10, atol=1e-14 * np.abs(I).max())
    # characteristic condition with a zero direction vector is the classical condition (4)
    Ic, _, _ = dg.rtm_backward(nglobal // 2, qT, hist, data, mode="classical", nglobal_total=nglobal)
    Iz, _, _ = dg.rtm_backward(nglobal // 2, qT, hist, data, updir=(0, 0, 0), nglobal_total=nglobal)
    assert np.allclose(Ic, Iz, rtol=1e-12, atol=0)
    assert not np.allclose(Ic, I, rtol=1e-3)
    # the classical image is the time integral of p_S p_R: compare with a fine trapezoid sum of
    # the stored nodal products on a half-step-refined run (third order vs first order)


def test_trace_history_layout_multirate():
    """Record count per level = nglobal*2^level + 1 (reading Q12); records equal the traces."""
    dg = _lts_setup(N=1, nlevels=3)
    dg.set_source(np.array([0.52, 0.47, 0.31]), f0=3.0, tp=0.1, amp=1.0)
    dg.receivers = dict(k=np.array([0]), row=np.zeros((1, dg.Np)), w=np.zeros((1, dg.Np)))
    data, hist, qT = dg.rtm_forward(3)
    for l in range(3):
        assert hist.records[l].shape[0] == 3 * 2 ** l + 1
        sel = hist.faces[l]
        assert np.all(dg.level[dg.bnd_k[sel]] == l)
    assert sum(len(s) for s in hist.faces) == np.sum(dg.bc == BC_ABSORBING)
    # the final record holds the traces of the final state
    qf = dg.traces_of(qT, np.arange(dg.K))
    for l in range(3):
        sel = hist.faces[l]
        assert np.array_equal(hist.records[l][-1], qf[dg.bnd_k[sel], dg.bnd_f[sel]])


def test_trapezoid_image_rule_closed_form():
    """(21) on fields linear in time over one step: integrand f(t) = (A + t rA)(B + t rB) is a quadratic, the
    trapezoid rule overshoots its integral by exactly rA rB dt^3 / 6, the AB-consistent rule (24) is exact."""
    from oracle.dgtd import DGOracle
    from workloads import box_tet_mesh
    etov, vx = box_tet_mesh(1, 1, 1)
    dg = DGOracle(2, etov, vx, default_bc=2)
    dg.set_model(np.ones(dg.K), np.ones(dg.K), 1, 0.15)
    rng = np.random.default_rng(5)
    FS, FR = dg.new_field(rng.standard_normal((dg.K, 4, dg.Np))), dg.new_field(rng.standard_normal((dg.K, 4, dg.Np)))
    rS, rR = rng.standard_normal((dg.K, 4, dg.Np)), rng.standard_normal((dg.K, 4, dg.Np))
    for F, r in ((FS, rS), (FR, rR)):
        F.hist[:] = r[None]                      # constant right-hand side: the field is linear in time
        F.nhist[:] = 3
    el = np.arange(dg.K)
    dt = 0.37
    A, B, rA, rB = FS.q[:, 0], FR.q[:, 0], rS[:, 0], rR[:, 0]
    exact = dt * A * B + dt ** 2 / 2 * (A * rB + B * rA) + dt ** 3 / 3 * rA * rB
    out = {}
    for mode in ("classical", "classical_trapezoid"):
        image = dict(I=np.zeros((dg.K, dg.Np)), mode=mode, updir=(0.0, 0.0, -1.0))
        dg.accumulate_image(image, FS, FR, el, dt)
        out[mode] = image["I"]
    assert np.abs(out["classical"] - exact).max() < 1e-12 * np.abs(exact).max()
    assert np.abs(out["classical_trapezoid"] - (exact + dt ** 3 / 6 * rA * rB)).max() < 1e-12 * np.abs(exact).max()
