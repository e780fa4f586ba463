"""ORACLE (test infrastructure, fp64, plain numpy) - the paper's nodal DGTD scheme, step by step.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this package.  It shares no code with the CUDA path (paper_1506_00907_b200/).  Nothing here is
blocked, fused or reordered beyond what the cited passage states.

PAPER.md = /root/reference/PAPER.md.  Implemented, in the paper's notation:
  * semi-discrete system (13)-(14) PAPER.md:113-118 with the penalties of (11)-(12) PAPER.md:100-102
    (factor 1/2 kept, reading Q2; single-valued face impedance, reading Q4; boundary
    exterior states, reading Q6);
  * point source (15) PAPER.md:122-128 scaled as in eq. (1) (reading Q5);
  * CFL time step PAPER.md:424, level structure PAPER.md:150-154 (reading Q9);
  * Algorithm 1 PAPER.md:222-242 with the update (18) and the coarse-neighbour half step (19),
    start-up by AB1, AB2 (reading Q7); backward in time with negative penalties PAPER.md:168;
  * boundary-trace capture / replay PAPER.md:70-72, 407 (reading Q12);
  * imaging conditions (4), (7) PAPER.md:49-65 integrated by the corrected formula (24)
    (readings Q1, Q1b).
  * LSERK4 (not in the paper; BASELINE.json config 1 only, reading Q8).

Parity unpinned (no value of the paper or of mathematics fixes them; only GPU-vs-oracle agreement and the
properties tested in tests/test_oracle_scheme.py hold): the AB start-up ramp by AB1, AB2 (reading Q7), the
reconstructed source wavefield and the image values at the configurations.

Array conventions: q[k, field, n] with field 0 = p, 1..3 = v_x, v_y, v_z; traces qf[k, f, i, 0] = p,
qf[k, f, i, 1] = n.v (outward normal of the owner); levels: 0 = coarsest (paper's
l = 1), L-1 = finest.
"""
import math

import numpy as np

from .reference_element import reference_element
from .mesh_geometry import (element_geometry, node_coordinates, connect_faces, match_face_nodes)
from .coefficients import ab_coefficients, ab_coefficients_exact, LSERK4_A, LSERK4_B, LSERK4_C

BC_INTERIOR, BC_FREE, BC_ABSORBING, BC_RIGID, BC_PRESCRIBED = 0, 1, 2, 3, 4


def ricker(t, f0, tp, amp=1.0):
    """Ricker pulse with peak frequency f0 and peak time tp."""
    a = (math.pi * f0 * (t - tp)) ** 2
    return amp * (1.0 - 2.0 * a) * math.exp(-a)


def ab_partial_weights(order, theta):
    """I_s(theta) = int_0^theta l_s for the order-`order` interpolant (22)."""
    from .coefficients import lagrange_on_past_steps, _poly_int, _poly_eval
    out = np.zeros(3)
    for s, p in enumerate(lagrange_on_past_steps(order)):
        out[s] = float(_poly_eval(_poly_int(p), theta))
    return out


class Wavefield:
    """q, the three most recent own right-hand sides (slot 0 newest), the exposed traces qf and the
    number of valid history entries per element (start-up order, reading Q7)."""

    def __init__(self, K, Np, Nfp):
        self.q = np.zeros((K, 4, Np))
        self.hist = np.zeros((3, K, 4, Np))
        self.nhist = np.zeros(K, dtype=np.int64)
        self.qf = np.zeros((K, 4, Nfp, 2))


class DGOracle:
    def __init__(self, N, EToV, VX, face_bc=None, default_bc=BC_ABSORBING):
        self.N = N
        self.ref = reference_element(N)
        self.Np, self.Nfp = self.ref.Np, self.ref.Nfp
        self.EToV = np.asarray(EToV, dtype=np.int64)
        self.VX = np.asarray(VX, dtype=np.float64)
        self.K = self.EToV.shape[0]
        self.geo = element_geometry(self.EToV, self.VX)
        if np.any(self.geo["J"] <= 0):
            raise ValueError("element with non-positive volume")
        self.EToE, self.EToF = connect_faces(self.EToV)
        self.mapP = match_face_nodes(self.ref, self.EToV, self.VX, self.EToE, self.EToF)
        bc = np.zeros((self.K, 4), dtype=np.int64)
        boundary = self.EToE < 0
        if face_bc is None:
            bc[boundary] = default_bc
        else:
            fb = np.asarray(face_bc).reshape(self.K, 4)
            bc[boundary] = np.where(fb[boundary] > 0, fb[boundary], default_bc)
        self.bc = bc
        # boundary-face list: all (k,f) with EToE = -1 in ascending (k,f) order
        kk, ff = np.nonzero(boundary)
        self.bnd_k, self.bnd_f = kk, ff
        self.bnd_index = np.full((self.K, 4), -1, dtype=np.int64)
        self.bnd_index[kk, ff] = np.arange(kk.size)
        self.X = node_coordinates(self.ref, self.EToV, self.VX)
        self.source = None
        self.receivers = None
        self.rho = None

    # -------------------------------------------------------------------------------------------
    # model, time step, levels
    # -------------------------------------------------------------------------------------------
    def set_model(self, rho, c, nlevels=1, cfl=0.15):
        self.rho = np.asarray(rho, dtype=np.float64).copy()
        self.c = np.asarray(c, dtype=np.float64).copy()
        self.Z = self.rho * self.c
        # local stable step, PAPER.md:424 and (17)
        self.dt_k = cfl * self.geo["ell"] / ((self.N + 1) ** 2 * self.c)
        self.dt_local = float(self.dt_k.min())
        self.nlevels = int(nlevels)
        self.level = assign_levels(self.dt_k, self.dt_local, self.EToE, self.nlevels)
        L = self.nlevels
        self.stride = 2 ** (L - 1 - self.level)             # fine steps per own step
        self.nlocal = 2 ** (L - 1)                           # fine steps per global step
        self.dt_global = self.dt_local * self.nlocal
        # elements that have a neighbour one level finer (coarse neighbours of Algorithm 1)
        nb_level = np.where(self.EToE >= 0, self.level[np.maximum(self.EToE, 0)], -1)
        self.has_finer_nbr = np.any(nb_level > self.level[:, None], axis=1)
        # single-valued face impedance (reading Q4)
        Znb = np.where(self.EToE >= 0, self.Z[np.maximum(self.EToE, 0)], self.Z[:, None])
        self.Zf = 0.5 * (self.Z[:, None] + Znb)

    # -------------------------------------------------------------------------------------------
    # point source / receivers  (eq. (15); reading Q5, Q11)
    # -------------------------------------------------------------------------------------------
    def locate(self, x0):
        """(element, r, s, t) of a point: lowest element id with all barycentrics >= -1e-10."""
        v0 = self.VX[self.EToV[:, 0]]
        d = np.asarray(x0, dtype=np.float64)[None, :] - v0                # [K,3]
        # (1+r, 1+s, 1+t)_j = sum_i (d r_j / d x_i) d_i
        rst1 = np.einsum("kij,ki->kj", self.geo["ginv"], d)
        lam = np.concatenate([1.0 - 0.5 * rst1.sum(axis=1, keepdims=True), 0.5 * rst1], axis=1)
        inside = np.all(lam >= -1e-10, axis=1)
        if not np.any(inside):
            raise ValueError("point outside the mesh")
        k = int(np.nonzero(inside)[0][0])
        r, s, t = rst1[k] - 1.0
        return k, r, s, t

    def point_weights(self, x0):
        """k, l(r0) (interpolation row) and w = M_k^-1 l(r0) = (1/J_k) M^-1 l(r0)."""
        k, r, s, t = self.locate(x0)
        ell = self.ref.interp_row(r, s, t)
        w = self.ref.Minv @ ell / self.geo["J"][k]
        return k, ell, w

    def set_source(self, x0, f0, tp, amp=1.0):
        k, ell, w = self.point_weights(x0)
        self.source = dict(k=k, w=w, f0=f0, tp=tp, amp=amp)

    def set_receivers(self, xr):
        xr = np.asarray(xr, dtype=np.float64).reshape(-1, 3)
        ks, rows, ws = [], [], []
        for x in xr:
            k, ell, w = self.point_weights(x)
            ks.append(k)
            rows.append(ell)
            ws.append(w)
        self.receivers = dict(k=np.array(ks), row=np.array(rows), w=np.array(ws))

    # -------------------------------------------------------------------------------------------
    # right-hand side
    # -------------------------------------------------------------------------------------------
    def traces_of(self, q, elems):
        """(p, n.v) at the face nodes of the given elements: [m,4,Nfp,2]."""
        return self.traces_from(q[elems], elems)

    def traces_from(self, qe, elems):
        """Same, from the nodal values qe [m,4,Np] of the elements `elems`."""
        fm = self.ref.Fmask                                     # [4,Nfp]
        out = np.empty((len(elems), 4, self.Nfp, 2))
        out[..., 0] = qe[:, 0][:, fm]
        n = self.geo["normals"][elems]                          # [m,4,3]
        vf = qe[:, 1:4][:, :, fm]                               # [m,3,4,Nfp]
        out[..., 1] = np.einsum("mfd,mdfi->mfi", n, vf)
        return out

    def rhs_volume(self, q, elems=None):
        """Volume terms of (13)-(14): -rho c^2 sum_ij g_ij D_j v_i and -(1/rho) sum_j g_ij D_j p."""
        if elems is None:
            elems = np.arange(self.K)
        ref = self.ref
        qe = q[elems]
        g = self.geo["ginv"][elems]                              # g[m,i,j] = d r_j / d x_i
        D = (ref.Dr, ref.Ds, ref.Dt)
        r = np.zeros_like(qe)
        dp = [qe[:, 0] @ D[j].T for j in range(3)]               # D_j p
        for i in range(3):
            for j in range(3):
                r[:, 0] -= g[:, i, j, None] * (qe[:, 1 + i] @ D[j].T)
                r[:, 1 + i] -= g[:, i, j, None] * dp[j]
        r[:, 0] *= (self.rho[elems] * self.c[elems] ** 2)[:, None]
        r[:, 1:4] /= self.rho[elems][:, None, None]
        return r

    def rhs_surface(self, q, qf, elems=None, direction=1, exterior=None):
        """Surface terms of (13)-(14): -sum_f g^sur_f L_f P_f with the penalties of (11)-(12).

        Interior values from q (the element is at its own time), neighbour values from the exposed
        traces qf (Alg. 3).  `exterior` [nbnd,Nfp,2] supplies (p+,
        n.v+) on prescribed faces (bc 4) and - when given - on absorbing faces too (trace replay).
        direction = -1 flips the sign of tau_p, tau_v."""
        if elems is None:
            elems = np.arange(self.K)
        own = self.traces_of(q, elems)                           # [m,4,Nfp,2]
        pm, nvm = own[..., 0], own[..., 1]
        nb = self.EToE[elems]                                    # [m,4]
        nbf = self.EToF[elems]
        safe = np.maximum(nb, 0)
        ext = np.take_along_axis(qf[safe, np.maximum(nbf, 0)], self.mapP[elems][..., None], axis=2)
        pp = ext[..., 0]
        nvp = -ext[..., 1]                                       # n- . v+ = -(n+ . v+)  (reading Q6b)
        bc = self.bc[elems]                                      # [m,4]
        dp = pp - pm
        dnv = nvp - nvm
        # boundary exterior states (reading Q6)
        free = (bc == BC_FREE)[..., None]
        rigid = (bc == BC_RIGID)[..., None]
        absorb = (bc == BC_ABSORBING)[..., None]
        presc = (bc == BC_PRESCRIBED)[..., None]
        dp = np.where(free, -2.0 * pm, dp)
        dnv = np.where(free, 0.0, dnv)
        dp = np.where(rigid, 0.0, dp)
        dnv = np.where(rigid, -2.0 * nvm, dnv)
        dp = np.where(absorb, -pm, dp)
        dnv = np.where(absorb, -nvm, dnv)
        if exterior is not None:
            b = np.maximum(self.bnd_index[elems], 0)             # [m,4]
            use = presc | absorb
            dp = np.where(use, exterior[b][..., 0] - pm, dp)
            dnv = np.where(use, exterior[b][..., 1] - nvm, dnv)
        elif np.any(presc):
            raise ValueError("prescribed-exterior faces need exterior values")
        Zf = self.Zf[elems][..., None]
        tau_v = direction * Zf
        tau_p = direction / Zf
        rho = self.rho[elems][:, None, None]
        c = self.c[elems][:, None, None]
        gs = self.geo["gsur"][elems][..., None]
        Pp = rho * c * c * 0.5 * (dnv - tau_p * dp) * gs          # [m,4,Nfp], already x J_f/J
        Pv = (1.0 / rho) * 0.5 * (dp - tau_v * dnv) * gs
        n = self.geo["normals"][elems]                            # [m,4,3]
        L = self.ref.LIFT                                         # [Np, 4*Nfp]
        m = len(elems)
        r = np.zeros((m, 4, self.Np))
        r[:, 0] = -(Pp.reshape(m, -1) @ L.T)
        for i in range(3):
            r[:, 1 + i] = -((n[:, :, i, None] * Pv).reshape(m, -1) @ L.T)
        return r

    def rhs(self, q, qf, t, elems=None, direction=1, exterior=None, source_on=True, injection=None):
        if elems is None:
            elems = np.arange(self.K)
        r = self.rhs_volume(q, elems) + self.rhs_surface(q, qf, elems, direction, exterior)
        pos = None
        if (source_on and self.source is not None) or injection is not None:
            pos = np.full(self.K, -1, dtype=np.int64)
            pos[elems] = np.arange(len(elems))
        if source_on and self.source is not None:
            s = self.source
            if pos[s["k"]] >= 0:
                r[pos[s["k"]], 0] += ricker(t, s["f0"], s["tp"], s["amp"]) * s["w"]
        if injection is not None:                                  # values d_r(t), [nr]
            rc = self.receivers
            here = pos[rc["k"]] >= 0
            np.add.at(r[:, 0], pos[rc["k"]][here], injection[here, None] * rc["w"][here])
        return r

    # -------------------------------------------------------------------------------------------
    # fields
    # -------------------------------------------------------------------------------------------
    def new_field(self, q0=None):
        F = Wavefield(self.K, self.Np, self.Nfp)
        if q0 is not None:
            F.q[...] = q0
        F.qf[...] = self.traces_of(F.q, np.arange(self.K))
        return F

    # -------------------------------------------------------------------------------------------
    # LSERK4 (reading Q8; config 1 only; single rate)
    # -------------------------------------------------------------------------------------------
    def run_lserk4(self, F, t0, dt, nsteps, exterior_fn=None):
        res = np.zeros_like(F.q)
        t = t0
        allk = np.arange(self.K)
        for _ in range(nsteps):
            for st in range(5):
                ts = t + LSERK4_C[st] * dt
                F.qf[...] = self.traces_of(F.q, allk)
                ext = exterior_fn(ts) if exterior_fn is not None else None
                r = self.rhs(F.q, F.qf, ts, exterior=ext)
                res = LSERK4_A[st] * res + dt * r
                F.q += LSERK4_B[st] * res
            t += dt
        F.qf[...] = self.traces_of(F.q, allk)
        return t

    # -------------------------------------------------------------------------------------------
    # Algorithm 1: multi-rate AB3, forward or backward, one or two wavefields
    # -------------------------------------------------------------------------------------------
    def run_mrab(self, fields, nglobal, t0, direction=1, *, source_on=(True,), exterior_fn=None,
                 capture=None, replay=None, record=None, injection=None, image=None,
                 first_fine_index=0):
        """Advance the wavefields in `fields` (list) by `nglobal` global steps from time t0.

        direction=+1 forward, -1 backward (time decreases, penalties negative).
        source_on[i]  : add the point source to field i.
        exterior_fn(t): exterior states for prescribed faces [nbnd,Nfp,2] (field 0 only).
        capture       : TraceHistory to WRITE boundary traces of field 0 into (forward RTM).
        replay        : TraceHistory to READ exterior states of field 0 from (backward RTM).
        record        : array [nr, nfine+1] receiving p(x_r) of field 0 at every fine time index.
        injection     : (field index, data [nr, nsamples]): d_r(t) w_r added to that field's r^p.
        image         : dict(I=[K,Np], mode="characteristic"|"classical", updir=[3]) accumulating
                        the imaging condition of fields[0] (source) x fields[1] (receivers).
        first_fine_index: absolute fine time index of t0 in FORWARD numbering (t = index*dt_local).
        """
        L = self.nlevels
        nloc = self.nlocal
        dtl = self.dt_local
        levels = [np.nonzero(self.level == l)[0] for l in range(L)]
        stride = [2 ** (L - 1 - l) for l in range(L)]
        coarse_nb = [np.nonzero((self.level == l) & self.has_finer_nbr)[0] for l in range(L)]
        nfine = nglobal * nloc
        for m in range(nfine):
            jabs = first_fine_index + direction * m          # absolute fine index of t_start
            t_start = t0 + direction * m * dtl
            # ---- right-hand sides of every element whose unknowns sit at t_start
            for l in range(L):
                if m % stride[l] != 0:
                    continue
                el = levels[l]
                if el.size == 0:
                    continue
                for fi, F in enumerate(fields):
                    ext = None
                    if fi == 0 and replay is not None:
                        ext = replay.exterior(l, jabs // stride[l])
                    elif fi == 0 and exterior_fn is not None:
                        ext = exterior_fn(t_start)
                    inj = None
                    if injection is not None and injection[0] == fi:
                        inj = injection[1][:, jabs]
                    r = self.rhs(F.q, F.qf, t_start, el, direction, ext,
                                 source_on=source_on[fi], injection=inj)
                    F.hist[2, el] = F.hist[1, el]
                    F.hist[1, el] = F.hist[0, el]
                    F.hist[0, el] = r
                    F.nhist[el] = np.minimum(F.nhist[el] + 1, 3)
                if capture is not None:
                    capture.store(l, jabs // stride[l], fields[0].qf)
            if record is not None:
                record[:, jabs] = self.sample_receivers(fields[0], m, stride, direction)
            # ---- updates (18) of the levels that land on t_new, finest first
            coarsest_updated = L
            for l in range(L - 1, -1, -1):
                if (m + 1) % stride[l] != 0:
                    continue
                coarsest_updated = l
                el = levels[l]
                if el.size == 0:
                    continue
                dts = direction * stride[l] * dtl                 # signed local step
                if image is not None:
                    self.accumulate_image(image, fields[0], fields[1], el, dts)
                for F in fields:
                    order = int(F.nhist[el[0]])
                    a = ab_coefficients(order)["a"]
                    F.q[el] += dts * (a[0] * F.hist[0, el] + a[1] * F.hist[1, el] + a[2] * F.hist[2, el])
                    F.qf[el] = self.traces_of(F.q, el)
            # ---- coarse neighbours that were not updated: half-step traces (19)
            lc = coarsest_updated - 1
            if 0 <= lc < L:
                el = coarse_nb[lc]
                if el.size:
                    dts = direction * stride[lc] * dtl
                    for F in fields:
                        order = int(F.nhist[el[0]])
                        b = ab_coefficients(order)["b"]
                        qh = F.q[el] + dts * (b[0] * F.hist[0, el] + b[1] * F.hist[1, el]
                                              + b[2] * F.hist[2, el])
                        F.qf[el] = self.traces_from(qh, el)
        jend = first_fine_index + direction * nfine
        if capture is not None:
            for l in range(L):
                capture.store(l, jend // stride[l], fields[0].qf)
        if record is not None:
            record[:, jend] = self.sample_receivers(fields[0], 0, stride, direction)
        return t0 + direction * nfine * dtl

    def sample_receivers(self, F, m, stride, direction):
        """p(x_r) at the current fine time: the nodal interpolant of the owning element; an element
        that is mid-step is evaluated with the AB interpolant (22) (reading Q13)."""
        rc = self.receivers
        out = np.empty(len(rc["k"]))
        for i, k in enumerate(rc["k"]):
            S = stride[self.level[k]]
            off = m % S
            p = F.q[k, 0]
            if off:
                wts = ab_partial_weights(int(F.nhist[k]), off / S)
                dts = direction * S * self.dt_local
                p = p + dts * (wts[0] * F.hist[0, k, 0] + wts[1] * F.hist[1, k, 0] + wts[2] * F.hist[2, k, 0])
            out[i] = rc["row"][i] @ p
        return out

    # -------------------------------------------------------------------------------------------
    # imaging (eqs (4), (7), (20)-(24); readings Q1, Q1b)
    # -------------------------------------------------------------------------------------------
    def accumulate_image(self, image, FS, FR, el, dts):
        order = int(FS.nhist[el[0]])
        co = ab_coefficients(order)
        trapezoid = image["mode"].endswith("_trapezoid")
        if image["mode"].startswith("characteristic"):
            e = np.asarray(image["updir"], dtype=np.float64)
            Z = self.Z[el][:, None]

            def down(x):      # q^- = p - c rho e.v   (source field)
                return x[:, 0] - Z * np.einsum("d,mdn->mn", e, x[:, 1:4])

            def up(x):        # q^+ = p + c rho e.v   (receiver field)
                return x[:, 0] + Z * np.einsum("d,mdn->mn", e, x[:, 1:4])
        else:
            def down(x):
                return x[:, 0]
            up = down
        A = down(FS.q[el])
        B = up(FR.q[el])
        rA = [down(FS.hist[s, el]) for s in range(3)]
        rB = [up(FR.hist[s, el]) for s in range(3)]
        acc = A * B
        for s in range(3):
            acc = acc + dts * co["abar"][s] * (A * rB[s] + B * rA[s])
            for s2 in range(3):
                acc = acc + dts * dts * co["C"][s, s2] * rA[s] * rB[s2]
        if trapezoid:
            # trapezoid rule (21) PAPER.md:178-180 (its printed "-" is a "+", reading Q1(v)): mean of the integrand at
            # the two ends of the local step; the values at the new time are the update (18) of the combinations
            A_new = A + dts * (co["a"][0] * rA[0] + co["a"][1] * rA[1] + co["a"][2] * rA[2])
            B_new = B + dts * (co["a"][0] * rB[0] + co["a"][1] * rB[1] + co["a"][2] * rB[2])
            acc = 0.5 * (A * B + A_new * B_new)
        image["I"][el] += abs(dts) * acc

    # -------------------------------------------------------------------------------------------
    # RTM driver (Fig. 1)
    # -------------------------------------------------------------------------------------------
    def rtm_forward(self, nglobal):
        """Source wavefield from rest; returns (data [nr, nfine+1] or None, TraceHistory, final q)."""
        F = self.new_field()
        hist = TraceHistory(self, nglobal)
        nfine = nglobal * self.nlocal
        data = np.zeros((len(self.receivers["k"]), nfine + 1)) if self.receivers else None
        self.run_mrab([F], nglobal, 0.0, 1, source_on=(True,), capture=hist, record=data,
                      first_fine_index=0)
        return data, hist, F.q.copy()

    def rtm_backward(self, nglobal, q_final, hist, data, updir=(0.0, 0.0, -1.0),
                     mode="characteristic", I=None, nglobal_total=None):
        """Source field reconstructed backward from q_final with trace replay, receiver field
        backward from rest with injection of `data`; image accumulated into I (returned)."""
        if nglobal_total is None:
            nglobal_total = nglobal
        FS = self.new_field(q_final)
        FR = self.new_field()
        if I is None:
            I = np.zeros((self.K, self.Np))
        image = dict(I=I, mode=mode, updir=updir)
        self.run_mrab([FS, FR], nglobal, nglobal_total * self.dt_global, -1,
                      source_on=(True, False), replay=hist, injection=(1, data), image=image,
                      first_fine_index=nglobal_total * self.nlocal)
        return I, FS, FR


class TraceHistory:
    """Boundary-trace storage (layout reading Q12): per level, record j holds
    (p, n.v) at the face nodes of the stored (absorbing) boundary faces owned by elements of that
    level, at time j * dt_level; faces in ascending (k,f) order."""

    def __init__(self, dg, nglobal):
        self.dg = dg
        L = dg.nlevels
        stored = dg.bc[dg.bnd_k, dg.bnd_f] == BC_ABSORBING
        self.faces = []          # per level: indices into the boundary-face list
        self.records = []
        for l in range(L):
            sel = np.nonzero(stored & (dg.level[dg.bnd_k] == l))[0]
            self.faces.append(sel)
            nrec = nglobal * 2 ** l + 1
            self.records.append(np.zeros((nrec, sel.size, dg.Nfp, 2)))

    def store(self, l, j, qf):
        sel = self.faces[l]
        self.records[l][j] = qf[self.dg.bnd_k[sel], self.dg.bnd_f[sel]]

    def exterior(self, l, j):
        """[nbnd,Nfp,2] exterior states (p+, n-.v+ = recorded n.v, reading Q6b) for level-l faces."""
        ext = np.zeros((self.dg.bnd_k.size, self.dg.Nfp, 2))
        ext[self.faces[l]] = self.records[l][j]
        return ext


def assign_levels(dt_k, dt_local, EToE, nlevels):
    """API level (0 = coarsest .. L-1 = finest) per element (reading Q9):
    raw exponent j = max{ j <= L-1 : 2^j dt_local <= dt_k }, then lowered until neighbouring
    elements differ by at most one level ("moved from coarse levels to finer levels")."""
    L = int(nlevels)
    K = dt_k.shape[0]
    j = np.zeros(K, dtype=np.int64)
    for e in range(1, L):
        j[(2.0 ** e) * dt_local <= dt_k] = e
    changed = True
    while changed:
        nbj = np.where(EToE >= 0, j[np.maximum(EToE, 0)], L + 10)
        cand = np.minimum(j, nbj.min(axis=1) + 1)
        changed = bool(np.any(cand != j))
        j = cand
    return ((L - 1) - j).astype(np.int32)
