"""Pins for the parts of oracle/dgtd.py that tests/test_oracle_scheme.py left unpinned (CPU only).

  * characteristic combinations q^-_S = p - Z e.v, q^+_R = p + Z e.v of eqs (7)-(8) PAPER.md:61-65, Z = rho c: a plane
    wave p = g(k.x - ct), v = k g/(rho c) travelling along -e has q^+ = 0 and q^- = 2p at every node, one along +e has
    q^- = 0 and q^+ = 2p (eqs (5)-(6) PAPER.md:55-57) -> the characteristic image of a down-going source field and an
    up-going receiver field is 4 x the classical image (4), that of the swapped pair vanishes; checked with rho != 1,
    c != 1 and oblique e, plus the bilinear expansion of (7) into four classical integrals;
  * ab_partial_weights / sample_receivers (reading Q13; interpolant (22) PAPER.md:184-188): I_s(1) = a_s and
    I_s(1/2) = b_s as printed in PAPER.md:161, 166; a field that is cubic in time is sampled exactly in mid-step;
  * sign convention Q1b: a backward-accumulated local-step integral equals the forward-time integral (20);
  * formula (24) keeps the third order of the fields, the trapezoid rule (21) does not;
  * Algorithm 1 with every element on one level is the plain AB3 recursion (18) written out with the printed weights.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle.dgtd import DGOracle, ab_partial_weights, BC_ABSORBING, BC_RIGID
from workloads import box_tet_mesh, graded_box_tet_mesh


def _plane_wave(dg, khat, rho, c, t=0.0):
    """Nodal values of p = g(k.x - ct), v = k g/(rho c) and of its time derivative."""
    g = lambda s: np.exp(-(s / 0.4) ** 2)
    dg_ds = lambda s: -2.0 * s / 0.4 ** 2 * np.exp(-(s / 0.4) ** 2)
    s = dg.X @ khat - 0.3 - c * t
    q = np.zeros((dg.K, 4, dg.Np))
    r = np.zeros((dg.K, 4, dg.Np))
    q[:, 0] = g(s)
    r[:, 0] = -c * dg_ds(s)
    for i in range(3):
        q[:, 1 + i] = khat[i] * g(s) / (rho * c)
        r[:, 1 + i] = khat[i] * (-c) * dg_ds(s) / (rho * c)
    return q, r


def _field_with_history(dg, khat, rho, c, dts):
    """Wavefield at t = 0 with the exact d/dt at t = 0, -dts, -2 dts in the three history slots."""
    q, _ = _plane_wave(dg, khat, rho, c, 0.0)
    F = dg.new_field(q)
    for s in range(3):
        F.hist[s] = _plane_wave(dg, khat, rho, c, -s * dts)[1]
    F.nhist[:] = 3
    return F


@pytest.mark.parametrize("e", [(0.0, 0.0, -1.0), (0.3, -0.2, -0.93), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0)])
def test_characteristic_fields_separate_up_and_down_going_plane_waves(e):
    e = np.asarray(e) / np.linalg.norm(e)
    rho, c = 2.2, 3.0                                   # Z = rho c = 6.6: rho or c alone fails the test
    etov, vx = box_tet_mesh(2, 2, 2, jitter=0.1, seed=3)
    dg = DGOracle(3, etov, vx, default_bc=BC_ABSORBING)
    dg.set_model(np.full(dg.K, rho), np.full(dg.K, c), 1, 0.15)
    el = np.arange(dg.K)
    dts = -0.01                                         # a backward local step, as in the RTM run
    down = _field_with_history(dg, -e, rho, c, dts)     # travels along -e: q^+ = 0, q^- = 2p
    up = _field_with_history(dg, +e, rho, c, dts)       # travels along +e: q^- = 0, q^+ = 2p

    def image(FS, FR, mode, updir=e):
        im = dict(I=np.zeros((dg.K, dg.Np)), mode=mode, updir=updir)
        dg.accumulate_image(im, FS, FR, el, dts)
        return im["I"]

    for suffix in ("", "_trapezoid"):
        Icl = image(down, up, "classical" + suffix)
        scale = np.abs(Icl).max()
        assert scale > 0
        # source down-going, receivers up-going: q^-_S q^+_R = (2 p_S)(2 p_R)
        assert np.abs(image(down, up, "characteristic" + suffix) - 4.0 * Icl).max() < 1e-12 * scale
        # source up-going, receivers down-going: both combinations vanish
        assert np.abs(image(up, down, "characteristic" + suffix)).max() < 1e-12 * scale
        # same-direction pairs: one factor vanishes
        assert np.abs(image(up, up, "characteristic" + suffix)).max() < 1e-12 * scale
        assert np.abs(image(down, down, "characteristic" + suffix)).max() < 1e-12 * scale
        # reversing e swaps the roles of q^+ and q^-
        assert np.abs(image(up, down, "characteristic" + suffix, updir=-e) - 4.0 * image(up, down, "classical" + suffix)
                      ).max() < 1e-12 * scale


def test_characteristic_image_is_the_bilinear_expansion_of_classical_integrals():
    """(7)-(8): int (p_S - Z e.v_S)(p_R + Z e.v_R) = I[p_S,p_R] + I[p_S,Z e.v_R] - I[Z e.v_S,p_R] - I[Z e.v_S,Z e.v_R],
    each term a classical integral (4) evaluated by the (Gauss-quadrature-pinned) classical branch on fields whose
    pressure slot holds the quantity; heterogeneous rho, c so that Z varies per element."""
    rng = np.random.default_rng(8)
    etov, vx = box_tet_mesh(2, 1, 1, jitter=0.1, seed=4)
    dg = DGOracle(2, etov, vx, default_bc=BC_ABSORBING)
    rho, c = rng.uniform(1.0, 2.5, dg.K), rng.uniform(1.5, 4.5, dg.K)
    dg.set_model(rho, c, 1, 0.15)
    el = np.arange(dg.K)
    e = np.array([0.3, -0.2, -0.93])
    e /= np.linalg.norm(e)

    def rand_field():
        F = dg.new_field(rng.standard_normal((dg.K, 4, dg.Np)))
        F.hist[:] = rng.standard_normal(F.hist.shape)
        F.nhist[:] = 3
        return F

    def pressure_only(F, which):
        """Field whose p slot is p (which = 0) or Z e.v (which = 1) of F, also in the history."""
        G = dg.new_field()
        Z = (rho * c)[:, None]
        if which == 0:
            G.q[:, 0] = F.q[:, 0]
            G.hist[:, :, 0] = F.hist[:, :, 0]
        else:
            G.q[:, 0] = Z * (e[0] * F.q[:, 1] + e[1] * F.q[:, 2] + e[2] * F.q[:, 3])
            G.hist[:, :, 0] = Z[None] * (e[0] * F.hist[:, :, 1] + e[1] * F.hist[:, :, 2] + e[2] * F.hist[:, :, 3])
        G.nhist[:] = 3
        return G

    FS, FR = rand_field(), rand_field()
    for dts in (0.02, -0.02):
        for suffix in ("", "_trapezoid"):
            def I(A, B, mode):
                im = dict(I=np.zeros((dg.K, dg.Np)), mode=mode + suffix, updir=e)
                dg.accumulate_image(im, A, B, el, dts)
                return im["I"]
            parts = (I(pressure_only(FS, 0), pressure_only(FR, 0), "classical")
                     + I(pressure_only(FS, 0), pressure_only(FR, 1), "classical")
                     - I(pressure_only(FS, 1), pressure_only(FR, 0), "classical")
                     - I(pressure_only(FS, 1), pressure_only(FR, 1), "classical"))
            Ich = I(FS, FR, "characteristic")
            assert np.abs(Ich - parts).max() < 1e-12 * np.abs(Ich).max()
            # e -> -e exchanges q^+ and q^-: the two cross terms change sign
            im = dict(I=np.zeros((dg.K, dg.Np)), mode="characteristic" + suffix, updir=-e)
            dg.accumulate_image(im, FS, FR, el, dts)
            cross = (I(pressure_only(FS, 0), pressure_only(FR, 1), "classical")
                     - I(pressure_only(FS, 1), pressure_only(FR, 0), "classical"))
            assert np.abs((Ich - im["I"]) - 2.0 * cross).max() < 1e-12 * np.abs(Ich).max()


def test_partial_weights_reproduce_the_printed_update_and_half_step_weights():
    """I_s(1) = a_s (eq (18)), I_s(1/2) = b_s (eq (19)), I_s(0) = 0; lower orders: AB1, AB2."""
    a3 = [Fraction(23, 12), Fraction(-16, 12), Fraction(5, 12)]
    b3 = [Fraction(17, 24), Fraction(-7, 24), Fraction(2, 24)]
    assert np.allclose(ab_partial_weights(3, 1.0), [float(x) for x in a3], rtol=0, atol=1e-15)
    assert np.allclose(ab_partial_weights(3, 0.5), [float(x) for x in b3], rtol=0, atol=1e-15)
    assert np.all(ab_partial_weights(3, 0.0) == 0.0)
    assert np.allclose(ab_partial_weights(2, 1.0), [1.5, -0.5, 0.0], rtol=0, atol=1e-15)
    assert np.allclose(ab_partial_weights(1, 0.25), [0.25, 0.0, 0.0], rtol=0, atol=1e-15)
    # quarter points (three-level runs sample at theta = 1/4, 3/4): closed form of int_0^theta l_s
    for th in (0.25, 0.75):
        l1 = th + 3 * th ** 2 / 4 + th ** 3 / 6          # l_1 = (t+1)(t+2)/2
        l2 = -(th ** 2 + th ** 3 / 3)                     # l_2 = -t(t+2)
        l3 = th ** 2 / 4 + th ** 3 / 6                    # l_3 = t(t+1)/2
        assert np.allclose(ab_partial_weights(3, th), [l1, l2, l3], rtol=0, atol=1e-15)


@pytest.mark.parametrize("direction", [1, -1])
def test_receivers_in_mid_step_sample_a_cubic_in_time_field_exactly(direction):
    """Reading Q13: a receiver owned by a level whose elements are mid-step is evaluated with the interpolant (22); for a
    field that is a cubic polynomial in time the right-hand side is quadratic, its three-point interpolant is exact, and
    so is the sample - at every fine offset of every level, in both time directions."""
    etov, vx = graded_box_tet_mesh(4, 4, 8, (1.0, 1.0, 1.0), band_center=0.5, band_width=0.2, max_ratio=4.0, seed=9,
                                   blob_sigma_cells=1.0)
    dg = DGOracle(2, etov, vx, default_bc=BC_ABSORBING)
    zc = vx[etov].mean(axis=1)[:, 2]
    dg.set_model(np.ones(dg.K), np.where((zc > 0.8) | (zc < 0.2), 1.0, 2.0), 3, 0.15)
    assert len(np.unique(dg.level)) == 3
    rng = np.random.default_rng(2)
    # three receivers per level, at the centroid of an element moved a little off it
    ks = np.concatenate([rng.choice(np.nonzero(dg.level == l)[0], 3, replace=False) for l in range(3)])
    xr = dg.VX[dg.EToV[ks]].mean(axis=1) + 1e-3
    dg.set_receivers(xr)
    assert np.array_equal(dg.level[dg.receivers["k"]], dg.level[ks])
    coef = rng.standard_normal((4, dg.K, dg.Np))                  # p(t) = c0 + c1 t + c2 t^2 + c3 t^3 per node
    p_of = lambda t: coef[0] + coef[1] * t + coef[2] * t ** 2 + coef[3] * t ** 3
    dp_of = lambda t: coef[1] + 2 * coef[2] * t + 3 * coef[3] * t ** 2
    stride = [4, 2, 1]
    t0 = 0.7
    F = dg.new_field()
    F.q[:, 0] = p_of(t0)
    F.nhist[:] = 3
    for k in range(dg.K):
        dtl = direction * stride[dg.level[k]] * dg.dt_local
        for s in range(3):
            F.hist[s, k, 0] = dp_of(t0 - s * dtl)[k]
    for m in range(4):
        got = dg.sample_receivers(F, m, stride, direction)
        for i, k in enumerate(dg.receivers["k"]):
            off = m % stride[dg.level[k]]
            want = dg.receivers["row"][i] @ p_of(t0 + direction * off * dg.dt_local)[k]
            assert abs(got[i] - want) < 1e-12 * max(1.0, abs(want)), (m, i, got[i], want)


def test_backward_accumulated_step_integral_equals_the_forward_one():
    """Reading Q1b: I = int_0^tf with dt > 0 (eqs (4), (7), (20) PAPER.md:49, 61, 174) whatever the run direction.  Fields
    linear in time on [ta, tb]: the forward step starts from the values at ta with dts = +dt, the backward step from the
    values at tb with dts = -dt; both give the closed form of int_ta^tb (A + t rA)(B + t rB) dt, which is positive for
    positive fields."""
    etov, vx = box_tet_mesh(1, 1, 1)
    dg = DGOracle(2, etov, vx, default_bc=BC_ABSORBING)
    dg.set_model(np.ones(dg.K), np.ones(dg.K), 1, 0.15)
    rng = np.random.default_rng(6)
    shape = (dg.K, 4, dg.Np)
    qS, qR = rng.uniform(1.0, 2.0, shape), rng.uniform(1.0, 2.0, shape)
    rS, rR = rng.uniform(0.1, 1.0, shape), rng.uniform(0.1, 1.0, shape)
    dt = 0.37
    A, B, rA, rB = qS[:, 0], qR[:, 0], rS[:, 0], rR[:, 0]
    exact = dt * A * B + dt ** 2 / 2 * (A * rB + B * rA) + dt ** 3 / 3 * rA * rB
    assert exact.min() > 0
    el = np.arange(dg.K)
    for mode, want in (("classical", exact), ("classical_trapezoid", exact + dt ** 3 / 6 * rA * rB)):
        out = {}
        for dts in (dt, -dt):
            FS = dg.new_field(qS if dts > 0 else qS + dt * rS)
            FR = dg.new_field(qR if dts > 0 else qR + dt * rR)
            for F, r in ((FS, rS), (FR, rR)):
                F.hist[:] = r[None]
                F.nhist[:] = 3
            im = dict(I=np.zeros((dg.K, dg.Np)), mode=mode, updir=(0.0, 0.0, -1.0))
            dg.accumulate_image(im, FS, FR, el, dts)
            out[dts] = im["I"]
        assert np.abs(out[dt] - want).max() < 1e-12 * want.max()
        assert np.abs(out[-dt] - want).max() < 1e-12 * want.max()


def test_formula_24_keeps_third_order_the_trapezoid_rule_does_not():
    """(24) 'keeps accuracy of numerical fields with an O(dt^3) numerical error', (21) does not.  Nodal
    signals A(t) = sin(w t + phi), B(t) = cos(v t + psi) with exact right-hand sides A', B' in the history slots,
    accumulated step by step over [0, T] (backward, as in the RTM run) against the closed-form integral."""
    etov, vx = box_tet_mesh(1, 1, 1)
    dg = DGOracle(1, etov, vx, default_bc=BC_ABSORBING)
    dg.set_model(np.ones(dg.K), np.ones(dg.K), 1, 0.15)
    rng = np.random.default_rng(12)
    w, v = rng.uniform(2.0, 4.0, (dg.K, dg.Np)), rng.uniform(2.0, 4.0, (dg.K, dg.Np))
    phi, psi = rng.uniform(0, 1, (dg.K, dg.Np)), rng.uniform(0, 1, (dg.K, dg.Np))
    T = 1.0
    # int_0^T sin(w t + phi) cos(v t + psi) dt = 1/2 int sin((w+v)t + phi+psi) + sin((w-v)t + phi-psi)
    def prim(t):
        return 0.5 * (-np.cos((w + v) * t + phi + psi) / (w + v) - np.cos((w - v) * t + phi - psi) / (w - v))
    exact = prim(T) - prim(0.0)
    el = np.arange(dg.K)
    errs = {"classical": [], "classical_trapezoid": []}
    for nsteps in (20, 40, 80):
        dt = T / nsteps
        for mode in errs:
            im = dict(I=np.zeros((dg.K, dg.Np)), mode=mode, updir=(0.0, 0.0, -1.0))
            FS, FR = dg.new_field(), dg.new_field()
            FS.nhist[:] = 3
            FR.nhist[:] = 3
            for n in range(nsteps):
                t = T - n * dt                           # step start; the step runs to t - dt
                FS.q[:, 0] = np.sin(w * t + phi)
                FR.q[:, 0] = np.cos(v * t + psi)
                for s in range(3):                       # own evaluations at t, t + dt, t + 2 dt (backward run)
                    FS.hist[s, :, 0] = w * np.cos(w * (t + s * dt) + phi)
                    FR.hist[s, :, 0] = -v * np.sin(v * (t + s * dt) + psi)
                dg.accumulate_image(im, FS, FR, el, -dt)
            errs[mode].append(np.abs(im["I"] - exact).max())
    e24, etr = errs["classical"], errs["classical_trapezoid"]
    assert np.log2(e24[0] / e24[1]) > 2.8 and np.log2(e24[1] / e24[2]) > 2.8, e24       # third order (or better)
    assert 1.7 < np.log2(etr[1] / etr[2]) < 2.3, etr                                      # second order at best
    assert e24[2] < 1e-2 * etr[2]


@pytest.mark.parametrize("level", [2, 1, 0])
def test_one_level_algorithm_1_is_the_plain_ab3_recursion(level):
    """All elements on one level of a three-level run (a uniform mesh puts every element on the finest level, step
    dt_local; forcing them onto the coarsest gives the step 4 dt_local): Algorithm 1 must reduce to
    q^{n+1} = q^n + dt (23/12 r^n - 16/12 r^{n-1} + 5/12 r^{n-2}) (eq (18)) with the AB1 / AB2
    start-up of reading Q7 - written out here with dg.rhs only."""
    etov, vx = box_tet_mesh(2, 2, 2)
    dg = DGOracle(2, etov, vx, default_bc=BC_RIGID)
    dg.set_model(np.ones(dg.K), np.ones(dg.K), 3, 0.15)
    assert np.all(dg.level == 2) and dg.nlocal == 4 and not dg.has_finer_nbr.any()
    dg.level[:] = level
    X = dg.X
    q0 = np.zeros((dg.K, 4, dg.Np))
    q0[:, 0] = np.cos(np.pi * X[..., 0]) * np.cos(np.pi * X[..., 1]) * np.cos(np.pi * X[..., 2])
    F = dg.new_field(q0)
    nglobal = 5
    dg.run_mrab([F], nglobal, 0.0, 1, source_on=(False,))
    dt = 2 ** (2 - level) * dg.dt_local
    nsteps = nglobal * 2 ** level
    q = q0.copy()
    hist = []
    weights = {1: [1.0], 2: [3.0 / 2, -1.0 / 2], 3: [23.0 / 12, -16.0 / 12, 5.0 / 12]}
    allk = np.arange(dg.K)
    for n in range(nsteps):
        qf = dg.traces_of(q, allk)
        hist.insert(0, dg.rhs(q, qf, n * dt, source_on=False))
        hist = hist[:3]
        wts = weights[len(hist)]
        q = q + dt * sum(wk * r for wk, r in zip(wts, hist))
    assert np.abs(F.q - q).max() <= 1e-14 * np.abs(q).max()
    # and a run asked for one level with the same step gives the same values
    dg1 = DGOracle(2, etov, vx, default_bc=BC_RIGID)
    dg1.set_model(np.ones(dg.K), np.ones(dg.K), 1, 0.15)
    dg1.dt_local = dg1.dt_global = dt
    G = dg1.new_field(q0)
    dg1.run_mrab([G], nsteps, 0.0, 1, source_on=(False,))
    assert np.abs(G.q - F.q).max() <= 1e-14 * np.abs(q).max()
