"""Domain decomposition of the (single- or multi-rate) scheme over several sub-domains:
set-up only - partition, local meshes, halo tables.  Every step of the path still runs in the library's kernels: a
sub-domain is an ordinary `DG` context whose cut faces are prescribed-exterior faces, and their exterior states are
fetched on the device from the neighbour's trace buffer by `dg_halo_pull` (k_halo) before every (fine) step.

    part = partition_elements(EToV, VX, nparts, weights)         # weighted recursive coordinate bisection
    dd = Decomposition(N, precision, EToV, VX, rho, c, part)     # one DG context per part, halo tables
    dd.bind_torch("cuda:0"); dd.dg_set_source(...); dd.dg_step(n); q = dd.dg_get_fields()
    dd.rtm_bind(nsteps, xr); data = dd.rtm_forward_shot(nsteps); dd.rtm_backward_shot(nsteps, data); I = dd.rtm_image_read()

The paper partitions with METIS, cell weights 2^(l-1) and keeps the finest cells off the cuts
(PAPER.md:387); METIS is not in this container: `partition_elements` is a weighted coordinate bisection that takes the same
weights and the same lumping of the finest cells with their neighbours.  With nlevels > 1 a sub-domain takes the levels of
the whole mesh (dg_set_model_levels), the exchange runs before every FINE step (dg_step_fine) and reads, per halo set, the
neighbour's current traces of that set's level or - the level being in mid-step - its half-step traces (eq (19)).  `Decomposition` keeps all sub-domains in one process (on one GPU their launches are ordered by the shared stream).
`RankDecomposition` is the one-process-per-sub-domain mode (one rank of torch.distributed = one sub-domain = one GPU): the
ranks exchange CUDA IPC handles of their workspaces once, after which the source pointer of `dg_halo_pull` is the peer
mapping of the neighbour's trace buffer - the loads of k_halo cross NVLink (or stay on the device when the ranks share a
GPU, which is how tests/test_decomp.py exercises it: this pool grants one GPU).  The ranks step in lock-step through a
host barrier per time step (no kernel waits on another).
"""
import numpy as np

from .binding import DG

BC_PRESCRIBED = 4


def face_neighbours(EToV):
    """[K][4] element behind each face (-1: boundary), faces matched by their sorted vertex triples (the order of the four
    faces of an element is the order of the vertex left out and plays no role for the partition)."""
    EToV = np.asarray(EToV)
    K = EToV.shape[0]
    tri = np.sort(np.stack([np.delete(EToV, v, axis=1) for v in range(4)], axis=1).reshape(4 * K, 3), axis=1)
    order = np.lexsort((tri[:, 2], tri[:, 1], tri[:, 0]))
    same = np.all(tri[order[1:]] == tri[order[:-1]], axis=1)
    nb = np.full(4 * K, -1, dtype=np.int64)
    a, b = order[:-1][same], order[1:][same]
    nb[a], nb[b] = b // 4, a // 4
    return nb.reshape(K, 4)


def lump_groups(lump, nb):
    """Group id per element (-1: none): every element flagged in `lump` together with its face neighbours; groups that
    share an element are merged ("lumping each finest element (or group of finest elements) with his
    neighbors")."""
    K = nb.shape[0]
    root = np.arange(K)

    def find(x):
        while root[x] != x:
            root[x] = root[root[x]]
            x = root[x]
        return x

    member = np.zeros(K, dtype=bool)
    for k in np.nonzero(lump)[0]:
        member[k] = True
        for k2 in nb[k]:
            if k2 >= 0:
                member[k2] = True
                ra, rb = find(k), find(int(k2))
                if ra != rb:
                    root[max(ra, rb)] = min(ra, rb)
    return np.array([find(k) if member[k] else -1 for k in range(K)], dtype=np.int64)


def partition_elements(EToV, VX, nparts, weights=None, lump=None):
    """Part id per element by recursive coordinate bisection of the element centroids along the longest axis, each cut
    balancing the summed weights (weight = local steps per global step of the cell).  lump: boolean mask of
    elements (the finest level's) that must not touch a cut: each is lumped with its face neighbours into one point
    before the bisection and separated afterwards, so that the fine steps that advance the finest level
    alone need no exchange."""
    K = EToV.shape[0]
    cen = VX[EToV].mean(axis=1)
    w = np.ones(K) if weights is None else np.asarray(weights, dtype=np.float64)
    if lump is not None and np.any(lump):
        grp = lump_groups(np.asarray(lump, dtype=bool), face_neighbours(EToV))
        for gid in np.unique(grp[grp >= 0]):
            m = grp == gid
            cen[m] = (cen[m] * w[m, None]).sum(axis=0) / w[m].sum()   # one point: a cut cannot separate its members
    part = np.zeros(K, dtype=np.int32)

    def split(idx, p0, n):
        if n == 1:
            part[idx] = p0
            return
        ext = cen[idx].max(axis=0) - cen[idx].min(axis=0)
        axis = int(np.argmax(ext))
        order = idx[np.lexsort((cen[idx, (axis + 2) % 3], cen[idx, (axis + 1) % 3], cen[idx, axis]))]
        nl = n // 2
        cw = np.cumsum(w[order])
        cut = int(np.searchsorted(cw, cw[-1] * nl / n)) + 1
        cut = min(max(cut, 1), len(order) - 1)
        same = np.all(cen[order[1:]] == cen[order[:-1]], axis=1)      # members of one lump are adjacent in `order`
        if same[cut - 1]:                                             # the cut falls inside a lump: move it to the nearer end
            lo, hi = cut, cut
            while lo > 1 and same[lo - 1]:
                lo -= 1
            lo = lo if not same[lo - 1] else 0
            while hi < len(order) - 1 and same[hi - 1]:
                hi += 1
            hi = hi if not same[hi - 1] else len(order)
            cands = [c for c in (lo, hi) if 1 <= c <= len(order) - 1]
            if cands:
                cut = min(cands, key=lambda c: abs(c - cut))
        split(order[:cut], p0, nl)
        split(order[cut:], p0 + nl, n - nl)

    split(np.arange(K), 0, int(nparts))
    return part


class Decomposition:
    """The sub-domains of one mesh as DG contexts with their halo tables.  Global arrays in, global arrays out."""

    def __init__(self, N, precision, EToV, VX, rho, c, part, default_bc=2, face_bc=None, cfl=0.15, only=None, nlevels=1,
                 fused=False):
        """only = p: bind / step sub-domain p alone (the others exist on the host for their slot tables).
        nlevels > 1: the multi-rate scheme; the levels and the finest step are those of the WHOLE mesh."""
        self.only = only
        self.fused = bool(fused)     # the step kernels read the halo faces' exterior states themselves (dg_halo_sources)
        self.nlevels, self.nlocal = int(nlevels), 1 << (int(nlevels) - 1)
        EToV = np.ascontiguousarray(EToV, dtype=np.int32)
        self.K, self.part = EToV.shape[0], np.asarray(part, dtype=np.int32)
        self.nparts = int(self.part.max()) + 1
        assert self.nparts <= 33, "a sub-domain has at most 32 halo sets (one per neighbour and level behind the cut)"
        # global connectivity and the global stable step from a host-only context of the whole mesh
        g = DG(N, precision, EToV, VX, face_bc=face_bc, default_bc=default_bc)
        g.dg_set_model(rho, c, self.nlevels, cfl)
        EToE, EToF, mapP = g.dg_get_connectivity()
        self.dt = g.dg_get_dt()[0]
        self.level = g.dg_get_levels()
        self._g = g                                                  # host-only context of the whole mesh (locates receivers)
        self.Np, self.Nfp = g.Np, g.Nfp
        self.elems = [np.nonzero(self.part == p)[0] for p in range(self.nparts)]
        local = np.full(self.K, -1, dtype=np.int64)
        for e in self.elems:
            local[e] = np.arange(e.size)
        self.local = local
        self.sub, self._halo = [], []
        Z = np.asarray(rho, dtype=np.float64) * np.asarray(c, dtype=np.float64)
        for p, e in enumerate(self.elems):
            verts, inv = np.unique(EToV[e], return_inverse=True)
            etov = inv.reshape(-1, 4).astype(np.int32)
            nb = EToE[e]                                              # [Kp][4] global neighbour or -1
            cut = (nb >= 0) & (self.part[np.maximum(nb, 0)] != p)
            fbc = np.full((e.size, 4), default_bc, dtype=np.int8) if face_bc is None else np.array(face_bc[e], dtype=np.int8)
            fbc[cut] = BC_PRESCRIBED
            s = DG(N, precision, etov, VX[verts], face_bc=fbc, default_bc=default_bc)
            bk, bf, bc = s.dg_get_boundary_faces()
            k2 = nb[bk, bf]                                           # global neighbour behind every boundary face
            halo = (k2 >= 0) & (bc == BC_PRESCRIBED)
            s.dg_set_model_levels(np.asarray(rho)[e], np.asarray(c)[e], self.nlevels, self.dt, self.level[e],
                                  np.where(halo, self.level[np.maximum(k2, 0)], -1))
            s.dg_set_exterior_impedance(np.where(halo, Z[np.maximum(k2, 0)], 0.0))
            self.sub.append(s)
            self._halo.append((bk, bf, k2, halo))
        self._tables(EToF, mapP)
        self._bound = False

    def _tables(self, EToF, mapP):
        slots = [s.dg_get_slots() for s in self.sub]
        self.sets = []                                               # per sub-domain: list of (neighbour part, tables),
        self.set_level = []                                          # one set per neighbour and level of the elements behind
        self.set_mine = []
        self.pulls = np.zeros(self.nlocal, dtype=np.int64)           # halo fetches enqueued per fine step of the cycle
        for p, s in enumerate(self.sub):
            bk, bf, k2, halo = self._halo[p]
            ge = self.elems[p][bk]                                    # global element of every boundary face
            sets, levels, mine = [], [], []
            for q in range(self.nparts):
                for lev in range(self.nlevels):
                    k2c = np.maximum(k2, 0)
                    sel = np.nonzero(halo & (self.part[k2c] == q) & (self.level[k2c] == lev))[0]
                    if q == p or sel.size == 0:
                        continue
                    f2 = EToF[ge[sel], bf[sel]]
                    rec = slots[q][self.local[k2[sel]]] * 4 + f2
                    pos = mapP[ge[sel], bf[sel]]                      # [nh][Nfp]: neighbour's face node at my node i
                    sets.append((q, sel.astype(np.int32), rec.astype(np.int64), pos.astype(np.int32)))
                    levels.append(lev)
                    mine.append(int(self.level[ge[sel]].max()))       # finest of MY elements on these faces
            assert len(sets) <= 32
            self.sets.append(sets)
            self.set_level.append(levels)
            self.set_mine.append(mine)

    # ---- memory, set-up
    def mine(self):
        return range(self.nparts) if self.only is None else (self.only,)

    def bind_torch(self, device="cuda:0"):
        for p in self.mine():
            s = self.sub[p]
            s.bind_torch(device)
            for i, (q, bnd, rec, pos) in enumerate(self.sets[p]):
                s.dg_set_halo(i, bnd, rec, pos)
        self._bound = True

    def dg_set_source(self, x0, f0, tp, amp=1.0):
        """The point source goes to the sub-domain that holds the element the whole mesh locates it in (reading Q11:
        lowest element id that contains the point); DGError if it lies outside the mesh."""
        self._g.dg_set_source(x0, f0, tp, amp)
        self.sub[int(self.part[self._g.dg_get_source()[0]])].dg_set_source(x0, f0, tp, amp)

    def dg_set_state(self, q, t0=0.0):
        for p, s in enumerate(self.sub):
            s.dg_set_state(q[self.elems[p]], t0)

    def dg_get_fields(self):
        q = np.empty((self.K, 4, self.Np))
        for p, s in enumerate(self.sub):
            q[self.elems[p]] = s.dg_get_fields()
        return q

    # ---- the step: every sub-domain pulls its halo, then every sub-domain advances one FINE step (Alg. 1)
    def first_level_starting_at(self, m):
        """Coarsest level whose step starts at fine step m of a global step (level l takes 2^(L-1-l) fine steps)."""
        lmin = self.nlevels - 1
        while lmin > 0 and m % (1 << (self.nlevels - lmin)) == 0:
            lmin -= 1
        return lmin

    def dg_step(self, nsteps):
        for _ in range(int(nsteps)):
            for m in range(self.nlocal):
                lmin = self.first_level_starting_at(m)
                tr = [s.dg_get_trace_levels() for s in self.sub]
                for p, s in enumerate(self.sub):
                    if self.fused:                               # no fetch launches: the step kernel reads these buffers
                        s.dg_halo_sources([tr[q][0][lev] if lev >= lmin else tr[q][1]
                                           for (q, _, _, _), lev in zip(self.sets[p], self.set_level[p])])
                        continue
                    for i, (q, _, _, _) in enumerate(self.sets[p]):
                        if self.set_mine[p][i] < lmin:          # none of my elements on these faces steps now (with the
                            continue                            # finest level off the cuts: no exchange at odd fine steps)
                        lev = self.set_level[p][i]              # traces at the time the fine levels have reached: the
                        s.dg_halo_pull(i, tr[q][0][lev] if lev >= lmin else tr[q][1])   # level's own, or its half-step ones
                        self.pulls[m] += 1
                for s in self.sub:
                    s.dg_step_fine(1)

    def launch_count(self):
        return sum(s.dg_get_launch_count() for s in self.sub)

    def close(self):
        for s in self.sub:
            s.close()
        self._g.close()

    # ---- RTM on the decomposed mesh: the source and the receiver run share the partition, so the imaging condition needs
    # no exchange; every sub-domain captures / replays the traces of ITS absorbing faces, records / injects
    # at ITS receivers and keeps ITS part of the image.  The exchange is the fused one (dg_halo_sources, rtm_halo_sources).
    def rtm_bind(self, nsteps, xr, device="cuda:0", spill_window=0):
        """Receivers (global list xr[nr][3]) to the sub-domains that contain them; trace histories for nsteps global steps
        (spill_window > 0: in pinned host memory behind a device ring of that many records, rtm_set_trace_spill)."""
        xr = np.asarray(xr, dtype=np.float64).reshape(-1, 3)
        self._g.dg_set_receivers(xr)
        self.rcv_sel = [np.nonzero(self.part[self._g.dg_get_receivers()[0]] == p)[0] for p in range(self.nparts)]
        self.nr = xr.shape[0]
        for p in self.mine():
            if self.rcv_sel[p].size:
                self.sub[p].dg_set_receivers(xr[self.rcv_sel[p]])
            if spill_window:
                self.sub[p].spill_traces_torch(nsteps, spill_window)
            self.sub[p].bind_history_torch(nsteps, device)

    def _fine_sources(self, m, tr, p):
        lmin = self.first_level_starting_at(m)
        return [tr[q][0][lev] if lev >= lmin else tr[q][1] for (q, _, _, _), lev in zip(self.sets[p], self.set_level[p])]

    def rtm_forward_shot(self, nsteps):
        """Forward phase in lock-step; returns the recorded signals data[nr][nfine + 1] in the order of rtm_bind's list."""
        total = nsteps * self.nlocal
        for s in self.sub:
            s.rtm_forward_part(nsteps, 0, 0)                          # initialise: the trace buffers are the phase's own now
        data = np.zeros((self.nr, total + 1))
        for j in range(total):
            tr = [s.rtm_get_trace_levels(0) for s in self.sub]
            for p, s in enumerate(self.sub):
                s.dg_halo_sources(self._fine_sources(j % self.nlocal, tr, p))
            for p, s in enumerate(self.sub):
                d = s.rtm_forward_part(nsteps, j, 1)
                if d is not None:
                    data[self.rcv_sel[p]] = d
        return data

    def rtm_backward_shot(self, nsteps, data, updir=(0.0, 0.0, -1.0), imaging=1, first_image_step=0):
        """Backward phase: both wavefields exchange their halo traces before every fine step, the image stays local."""
        total = nsteps * self.nlocal
        for p, s in enumerate(self.sub):
            s.rtm_backward_part(nsteps, data[self.rcv_sel[p]] if self.rcv_sel[p].size else None, 0, 0, updir, imaging,
                                first_image_step)
        for j in range(total):
            trF = [s.rtm_get_trace_levels(0) for s in self.sub]
            trR = [s.rtm_get_trace_levels(1) for s in self.sub]
            for p, s in enumerate(self.sub):
                s.dg_halo_sources(self._fine_sources(j % self.nlocal, trF, p))
                s.rtm_halo_sources(self._fine_sources(j % self.nlocal, trR, p))
            for s in self.sub:
                s.rtm_backward_part(nsteps, None, j, 1, updir, imaging, first_image_step)

    def rtm_image_read(self):
        img = np.empty((self.K, self.Np))
        for p, s in enumerate(self.sub):
            img[self.elems[p]] = s.rtm_image_read()
        return img


class RankDecomposition(Decomposition):
    """One sub-domain per torch.distributed rank.  Every rank builds the host side of all sub-domains (their slot tables
    are needed for the halo tables), binds its own, and maps the workspaces of its neighbours through CUDA IPC; the
    trace buffer of a neighbour is then addressed as (mapped workspace base + the offset that neighbour reports)."""

    def __init__(self, dist, *args, **kw):
        self.dist, self.rank = dist, dist.get_rank()
        super().__init__(*args, only=self.rank, **kw)
        assert self.nparts == dist.get_world_size(), "one sub-domain per rank"

    def bind_torch(self, device="cuda:0"):
        import torch
        from torch.multiprocessing.reductions import reduce_tensor
        super().bind_torch(device)
        me = self.sub[self.rank]
        self._device = device
        handles = [None] * self.nparts
        self.dist.all_gather_object(handles, reduce_tensor(me._ws))       # (rebuild function, arguments) per rank
        self._peer = {}
        for q, _, _, _ in self.sets[self.rank]:
            fn, a = handles[q]
            self._peer[q] = fn(*a)                                        # the neighbour's workspace tensor, mapped here
            self._enable_peer(self._peer[q])
        self._buf_off = {0: self._gather_buffer_offsets(0, me._ws)}
        self.dist.barrier()

    def _gather_buffer_offsets(self, field, tensor):
        """Once: every rank's two alternating trace buffers and half-step buffer as offsets inside its shared tensor."""
        me = self.sub[self.rank]
        self._my_bufs = getattr(self, "_my_bufs", {})
        self._my_bufs[field] = me.dg_get_trace_buffers(field)
        offs = [None] * self.nparts
        self.dist.all_gather_object(offs, [int(b - tensor.data_ptr()) for b in self._my_bufs[field]])
        return offs

    def _current_offsets(self, field):
        """Per rank ([offset of the current buffer of level l], offset of the half-step buffer).  Sub-domains in lock-step
        alternate their buffers alike: the neighbour's current buffer of a level is the one with MY parity of that level.
        The barrier orders this fine step after every rank's previous one."""
        me = self.sub[self.rank]
        cur = (me.dg_get_trace_levels() if field == 0 else me.rtm_get_trace_levels(field))[0]
        par = [0 if c == self._my_bufs[field][0] else 1 for c in cur]
        self.dist.barrier()
        return [([o[p] for p in par], o[2]) for o in self._buf_off[field]]

    def _enable_peer(self, t):
        """A mapping that lives on another GPU is read by MY kernels through NVLink: that needs peer access from my device,
        which torch switches on with the first device-to-device copy between the pair (one GPU in this pool: not exercised)."""
        import torch
        mine = torch.device(self._device)
        if t.device != mine:
            torch.empty(1, dtype=t.dtype, device=mine).copy_(t.view(-1)[:1])

    def _trace_offsets(self):
        return self._current_offsets(0)

    def dg_step(self, nsteps):
        import torch
        me = self.sub[self.rank]
        for _ in range(int(nsteps)):
            for m in range(self.nlocal):
                lmin = self.first_level_starting_at(m)
                offs = self._trace_offsets()        # (a barrier: this step comes after every rank's previous one)
                if self.fused:                      # my step kernel reads the neighbours' buffers; they write the OTHER ones
                    me.dg_halo_sources([self._peer[q].data_ptr() + (offs[q][0][lev] if lev >= lmin else offs[q][1])
                                        for (q, _, _, _), lev in zip(self.sets[self.rank], self.set_level[self.rank])])
                    me.dg_step_fine(1)
                    torch.cuda.synchronize(self._device)    # my reads and my new traces are complete before the next barrier
                    continue
                for i, (q, _, _, _) in enumerate(self.sets[self.rank]):
                    if self.set_mine[self.rank][i] < lmin:
                        continue
                    lev = self.set_level[self.rank][i]
                    self.pulls[m] += 1
                    me.dg_halo_pull(i, self._peer[q].data_ptr() + (offs[q][0][lev] if lev >= lmin else offs[q][1]))
                torch.cuda.synchronize(self._device)    # my fetches have read the neighbours' traces ...
                self.dist.barrier()                     # ... on every rank, before anybody's step overwrites them
                me.dg_step_fine(1)
                torch.cuda.synchronize(self._device)    # my new traces are complete before the next barrier returns

    def dg_set_state(self, q, t0=0.0):
        self.sub[self.rank].dg_set_state(q[self.elems[self.rank]], t0)

    # ---- RTM, one process per sub-domain: the fused exchange for both wavefields, a host barrier per fine step
    def _field_offsets(self, field):
        return self._current_offsets(field)

    def _peer_sources(self, m, offs, peer):
        lmin = self.first_level_starting_at(m)
        return [peer[q].data_ptr() + (offs[q][0][lev] if lev >= lmin else offs[q][1])
                for (q, _, _, _), lev in zip(self.sets[self.rank], self.set_level[self.rank])]

    def rtm_bind(self, nsteps, xr, device="cuda:0", spill_window=0):
        from torch.multiprocessing.reductions import reduce_tensor
        super().rtm_bind(nsteps, xr, device, spill_window)
        handles = [None] * self.nparts
        self.dist.all_gather_object(handles, reduce_tensor(self.sub[self.rank]._hist))
        self._peer_hist = {}
        for q, _, _, _ in self.sets[self.rank]:
            fn, a = handles[q]
            self._peer_hist[q] = fn(*a)
            self._enable_peer(self._peer_hist[q])
        self._buf_off[1] = self._gather_buffer_offsets(1, self.sub[self.rank]._hist)
        self.dist.barrier()

    def rtm_forward_shot(self, nsteps):
        import torch
        me, total = self.sub[self.rank], nsteps * self.nlocal
        me.rtm_forward_part(nsteps, 0, 0)
        torch.cuda.synchronize(self._device)
        mine = None
        for j in range(total):
            offs = self._field_offsets(0)               # orders this step after every rank's previous one
            me.dg_halo_sources(self._peer_sources(j % self.nlocal, offs, self._peer))
            mine = me.rtm_forward_part(nsteps, j, 1)
            torch.cuda.synchronize(self._device)
        parts = [None] * self.nparts
        self.dist.all_gather_object(parts, mine)
        data = np.zeros((self.nr, total + 1))
        for p in range(self.nparts):
            if parts[p] is not None:
                data[self.rcv_sel[p]] = parts[p]
        return data

    def rtm_backward_shot(self, nsteps, data, updir=(0.0, 0.0, -1.0), imaging=1, first_image_step=0):
        import torch
        me, total, sel = self.sub[self.rank], nsteps * self.nlocal, self.rcv_sel[self.rank]
        me.rtm_backward_part(nsteps, data[sel] if sel.size else None, 0, 0, updir, imaging, first_image_step)
        torch.cuda.synchronize(self._device)
        for j in range(total):
            offF, offR = self._field_offsets(0), self._field_offsets(1)
            me.dg_halo_sources(self._peer_sources(j % self.nlocal, offF, self._peer))
            me.rtm_halo_sources(self._peer_sources(j % self.nlocal, offR, self._peer_hist))
            me.rtm_backward_part(nsteps, None, j, 1, updir, imaging, first_image_step)
            torch.cuda.synchronize(self._device)

    def rtm_image_read(self):
        parts = [None] * self.nparts
        self.dist.all_gather_object(parts, self.sub[self.rank].rtm_image_read())
        img = np.empty((self.K, self.Np))
        for p in range(self.nparts):
            img[self.elems[p]] = parts[p]
        return img

    def dg_get_fields(self):
        """Global field on every rank (host all-gather of the sub-domain fields)."""
        mine = self.sub[self.rank].dg_get_fields()
        parts = [None] * self.nparts
        self.dist.all_gather_object(parts, mine)
        q = np.empty((self.K, 4, self.Np))
        for p in range(self.nparts):
            q[self.elems[p]] = parts[p]
        return q

    def launch_count(self):
        return self.sub[self.rank].dg_get_launch_count()
