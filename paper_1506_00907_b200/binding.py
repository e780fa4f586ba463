"""Thin ctypes binding of libdgrtm.so (include/dgrtm.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch supplies device memory
(uint8 tensors) and the stream, nothing else.  There is no CPU fallback: if the library is missing
the import of this module fails.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdgrtm.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libdgrtm.so is not built: run `python -m paper_1506_00907_b200.build` "
        "(there is no CPU fallback for the DGTD hot path)")
_lib = C.CDLL(LIB_PATH)

DG_OK = 0
DG_ERR_ARG, DG_ERR_MESH, DG_ERR_STATE, DG_ERR_CUDA, DG_ERR_NOMEM, DG_ERR_UNSUPPORTED = -1, -2, -3, -4, -5, -6
DG_BC_FREE, DG_BC_ABSORBING, DG_BC_RIGID, DG_BC_PRESCRIBED = 1, 2, 3, 4
DG_INTEGRATOR_AB3, DG_INTEGRATOR_LSERK4 = 0, 1
DG_WAVELET_RICKER = 0
DG_IMAGING_CLASSICAL, DG_IMAGING_CHARACTERISTIC = 0, 1
DG_IMAGING_CLASSICAL_TRAPEZOID, DG_IMAGING_CHARACTERISTIC_TRAPEZOID = 2, 3
DG_RHS_VOLUME, DG_RHS_SURFACE, DG_RHS_TOTAL = 0, 1, 2
KERNEL_CLASSES = ("rhs", "update", "halo", "image_update", "source", "record", "inject", "capture", "rk", "step", "step_image")

_vp, _i, _i64, _d, _sz = C.c_void_p, C.c_int, C.c_int64, C.c_double, C.c_size_t
_pd = C.POINTER(C.c_double)
_pi32 = C.POINTER(C.c_int32)
_pi8 = C.POINTER(C.c_int8)
_pi64 = C.POINTER(C.c_int64)
_pint = C.POINTER(C.c_int)
_psz = C.POINTER(C.c_size_t)

# name -> (restype, argtypes): the complete export list of include/dgrtm.h
SIGNATURES = {
    "dg_version": (C.c_char_p, []),
    "dg_last_error": (C.c_char_p, [_vp]),
    "dg_mesh_create": (_i, [C.POINTER(_vp), _i, _i, _i64, _i64, _pi32, _pd, _pi8, _i]),
    "dg_destroy": (None, [_vp]),
    "dg_set_model": (_i, [_vp, _pd, _pd, _i, _d]),
    "dg_set_integrator": (_i, [_vp, _i]),
    "dg_set_dt": (_i, [_vp, _d]),
    "dg_set_source": (_i, [_vp, _pd, _i, _d, _d, _d]),
    "dg_set_receivers": (_i, [_vp, _i64, _pd]),
    "dg_workspace_bytes": (_i, [_vp, _psz]),
    "dg_bind_workspace": (_i, [_vp, _vp, _sz, _vp]),
    "dg_set_state": (_i, [_vp, _pd, _d]),
    "dg_step": (_i, [_vp, _i]),
    "dg_set_exterior": (_i, [_vp, _pd]),
    "dg_step_lserk4_static": (_i, [_vp, _i]),
    "dg_static_scratch_bytes": (_i, [C.POINTER(_sz)]),
    "dg_set_exterior_impedance": (_i, [_vp, _pd]),
    "dg_get_slots": (_i, [_vp, _pi64]),
    "dg_get_trace_device": (_i, [_vp, C.POINTER(_vp), C.POINTER(_sz)]),
    "dg_set_halo": (_i, [_vp, _i, _i64, _pi32, _pi64, _pi32]),
    "dg_halo_pull": (_i, [_vp, _i, _vp]),
    "dg_set_model_levels": (_i, [_vp, _pd, _pd, _i, _d, _pi32, _pi32]),
    "dg_step_fine": (_i, [_vp, _i]),
    "dg_get_trace_levels": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_sz)]),
    "dg_halo_sources": (_i, [_vp, _i, C.POINTER(_vp)]),
    "dg_get_trace_buffers": (_i, [_vp, _i, C.POINTER(_vp), C.POINTER(_sz)]),
    "rtm_set_receiver_capacity": (_i, [_vp, _i64]),
    "rtm_set_spill_packing": (_i, [_vp, _i]),
    "rtm_spill_bytes": (_i, [_vp, _i, C.POINTER(_sz)]),
    "rtm_set_trace_spill": (_i, [_vp, _vp, _sz, _i]),
    "rtm_history_bytes": (_i, [_vp, _i, _psz]),
    "rtm_bind_history": (_i, [_vp, _vp, _sz]),
    "rtm_forward_shot": (_i, [_vp, _i, _pd]),
    "rtm_backward_shot": (_i, [_vp, _i, _pd, _pd, _i, _i64]),
    "rtm_forward_part": (_i, [_vp, _i, _i64, _i64, _pd]),
    "rtm_backward_part": (_i, [_vp, _i, _pd, _pd, _i, _i64, _i64, _i64]),
    "rtm_get_trace_levels": (_i, [_vp, _i, C.POINTER(_vp), C.POINTER(_vp), C.POINTER(_sz)]),
    "rtm_halo_sources": (_i, [_vp, _i, C.POINTER(_vp)]),
    "rtm_image_read": (_i, [_vp, _pd]),
    "rtm_image_zero": (_i, [_vp]),
    "rtm_image_device": (_i, [_vp, C.POINTER(_vp), _psz]),
    "dg_get_sizes": (_i, [_vp, _pi64, _pint, _pint, _pi64, _pi64]),
    "dg_get_nodes": (_i, [_vp, _pd, _pd, _pd]),
    "dg_get_operators": (_i, [_vp, _pd, _pd, _pd, _pd, _pi32]),
    "dg_get_connectivity": (_i, [_vp, _pi32, _pi32, _pi32]),
    "dg_get_boundary_faces": (_i, [_vp, _pi32, _pi32, _pi32]),
    "dg_get_geometry": (_i, [_vp, _pd, _pd, _pd, _pd, _pd]),
    "dg_get_levels": (_i, [_vp, _pi32]),
    "dg_get_dt": (_i, [_vp, _pd, _pint]),
    "dg_get_time": (_i, [_vp, _pd]),
    "dg_get_source": (_i, [_vp, _pi32, _pd]),
    "dg_get_receivers": (_i, [_vp, _pi32, _pd, _pd]),
    "dg_get_fields": (_i, [_vp, _pd]),
    "dg_get_traces": (_i, [_vp, _pd]),
    "dg_get_rhs": (_i, [_vp, _i, _i, _pd]),
    "rtm_get_trace_index": (_i, [_vp, _i, _pi64, _pi64, _pi32]),
    "rtm_get_traces": (_i, [_vp, _i, _i64, _pd]),
    "rtm_get_fields": (_i, [_vp, _i, _pd]),
    "dg_get_launch_count": (_i, [_vp, _pi64]),
    "dg_set_profiling": (_i, [_vp, _i]),
    "dg_get_kernel_times": (_i, [_vp, _pd, _pi64]),
    "dg_bench_kernel": (_i, [_vp, _i, _i]),
    "dg_measure_fma": (_i, [_i, _vp, _sz, _vp, _pd]),
}
for _name, (_res, _args) in SIGNATURES.items():
    _fn = getattr(_lib, _name)
    _fn.restype = _res
    _fn.argtypes = _args


class DGError(RuntimeError):
    def __init__(self, code, message):
        super().__init__("libdgrtm error %d: %s" % (code, message))
        self.code = code


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def dg_static_scratch_bytes():
    n = _sz()
    rc = _lib.dg_static_scratch_bytes(C.byref(n))
    assert rc == DG_OK
    return n.value


def _ptr(a, typ):
    return None if a is None else a.ctypes.data_as(typ)


class DG:
    """One dg_ctx.  Method names are the C entry points without the dg_/rtm_ split removed:
    dg_mesh_create is the constructor; every other call is a method of the same name."""

    def __init__(self, N, precision, EToV, VX, face_bc=None, default_bc=DG_BC_ABSORBING):
        etov = np.ascontiguousarray(EToV, dtype=np.int32)
        vx = _f64(VX)
        fb = None if face_bc is None else np.ascontiguousarray(face_bc, dtype=np.int8)
        self._h = _vp()
        rc = _lib.dg_mesh_create(C.byref(self._h), int(N), int(precision), etov.shape[0], vx.shape[0],
                                 _ptr(etov, _pi32), _ptr(vx, _pd), _ptr(fb, _pi8), int(default_bc))
        if rc != DG_OK:
            raise DGError(rc, (_lib.dg_last_error(None) or b"").decode())
        self.N, self.precision = int(N), int(precision)
        K, Np, Nfp, nbnd, nr = _i64(), _i(), _i(), _i64(), _i64()
        _lib.dg_get_sizes(self._h, C.byref(K), C.byref(Np), C.byref(Nfp), C.byref(nbnd), C.byref(nr))
        self.K, self.Np, self.Nfp, self.nbnd = K.value, Np.value, Nfp.value, nbnd.value
        self.nr = 0
        self._ws = None
        self._hist = None

    def close(self):
        if getattr(self, "_h", None):
            _lib.dg_destroy(self._h)
            self._h = None
        self._ws = None
        self._hist = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != DG_OK:
            raise DGError(rc, (_lib.dg_last_error(self._h) or b"").decode())

    # ---- setup
    def dg_set_model(self, rho, c, nlevels=1, cfl=0.15):
        rho, c = _f64(rho), _f64(c)
        assert rho.shape == (self.K,) and c.shape == (self.K,)
        self._ck(_lib.dg_set_model(self._h, _ptr(rho, _pd), _ptr(c, _pd), int(nlevels), float(cfl)))

    def dg_set_integrator(self, integrator):
        self._ck(_lib.dg_set_integrator(self._h, int(integrator)))

    def dg_set_dt(self, dt_local):
        self._ck(_lib.dg_set_dt(self._h, float(dt_local)))

    def dg_set_source(self, x0, f0, tp, amp=1.0, wavelet=DG_WAVELET_RICKER):
        x0 = _f64(x0)
        self._ck(_lib.dg_set_source(self._h, _ptr(x0, _pd), int(wavelet), float(f0), float(tp), float(amp)))

    def dg_set_receivers(self, xr):
        xr = _f64(xr).reshape(-1, 3)
        self._ck(_lib.dg_set_receivers(self._h, xr.shape[0], _ptr(xr, _pd)))
        self.nr = xr.shape[0]

    def dg_workspace_bytes(self):
        n = _sz()
        self._ck(_lib.dg_workspace_bytes(self._h, C.byref(n)))
        return n.value

    def dg_bind_workspace(self, dptr, nbytes, stream=0):
        self._ck(_lib.dg_bind_workspace(self._h, _vp(dptr), nbytes, _vp(stream)))

    def bind_torch(self, device="cuda:0", stream=None):
        """Allocates the workspace as a torch uint8 tensor and binds it with torch's current stream."""
        import torch
        n = self.dg_workspace_bytes()
        self._ws = torch.empty(n + 256, dtype=torch.uint8, device=device)
        base = (self._ws.data_ptr() + 255) & ~255
        s = stream if stream is not None else torch.cuda.current_stream(device).cuda_stream
        self.dg_bind_workspace(base, n, s)
        return n

    # ---- stepping
    def dg_set_state(self, q, t0=0.0):
        q = _f64(q)
        assert q.shape == (self.K, 4, self.Np)
        self._ck(_lib.dg_set_state(self._h, _ptr(q, _pd), float(t0)))

    def dg_step(self, nsteps):
        self._ck(_lib.dg_step(self._h, int(nsteps)))

    def dg_step_lserk4_static(self, nsteps):
        """LSERK4 steps with the stage residual in the library's static device array (no allocation; <= 8 MiB of state)."""
        self._ck(_lib.dg_step_lserk4_static(self._h, int(nsteps)))

    def dg_set_exterior(self, ext):
        ext = _f64(ext)
        assert ext.shape == (self.nbnd, self.Nfp, 2)
        self._ck(_lib.dg_set_exterior(self._h, _ptr(ext, _pd)))

    # ---- domain decomposition (halo faces)
    def dg_set_exterior_impedance(self, Zext):
        Zext = None if Zext is None else _f64(Zext)
        assert Zext is None or Zext.shape == (self.nbnd,)
        self._ck(_lib.dg_set_exterior_impedance(self._h, _ptr(Zext, _pd)))

    def dg_get_slots(self):
        s = np.empty(self.K, dtype=np.int64)
        self._ck(_lib.dg_get_slots(self._h, _ptr(s, _pi64)))
        return s

    def dg_get_trace_device(self):
        p, n = _vp(), _sz()
        self._ck(_lib.dg_get_trace_device(self._h, C.byref(p), C.byref(n)))
        return p.value, n.value

    def dg_set_halo(self, halo_set, bnd_index, src_record, src_pos):
        bnd_index = np.ascontiguousarray(bnd_index, dtype=np.int32)
        src_record = np.ascontiguousarray(src_record, dtype=np.int64)
        src_pos = np.ascontiguousarray(src_pos, dtype=np.int32)
        assert src_record.shape == bnd_index.shape and src_pos.shape == (bnd_index.size, self.Nfp)
        self._ck(_lib.dg_set_halo(self._h, int(halo_set), int(bnd_index.size), _ptr(bnd_index, _pi32), _ptr(src_record, _pi64),
                                  _ptr(src_pos, _pi32)))

    def dg_halo_pull(self, halo_set, src_trace_device):
        self._ck(_lib.dg_halo_pull(self._h, int(halo_set), _vp(src_trace_device)))

    def dg_set_model_levels(self, rho, c, nlevels, dt_local, level, bnd_level=None):
        rho, c = _f64(rho), _f64(c)
        level = np.ascontiguousarray(level, dtype=np.int32)
        bnd_level = None if bnd_level is None else np.ascontiguousarray(bnd_level, dtype=np.int32)
        assert rho.shape == (self.K,) and c.shape == (self.K,) and level.shape == (self.K,)
        assert bnd_level is None or bnd_level.shape == (self.nbnd,)
        self._ck(_lib.dg_set_model_levels(self._h, _ptr(rho, _pd), _ptr(c, _pd), int(nlevels), float(dt_local),
                                          _ptr(level, _pi32), _ptr(bnd_level, _pi32)))

    def dg_step_fine(self, nfine):
        self._ck(_lib.dg_step_fine(self._h, int(nfine)))

    def dg_get_trace_levels(self):
        """([device pointer of the current traces of level l], device pointer of the half-step traces, bytes of each)."""
        L = int(self.dg_get_dt()[1]).bit_length()                     # nlocal = 2^(L-1) fine steps per global step
        cur, half, n = (_vp * 8)(), _vp(), _sz()
        self._ck(_lib.dg_get_trace_levels(self._h, cur, C.byref(half), C.byref(n)))
        return [cur[l] for l in range(L)], half.value, n.value

    def dg_get_trace_buffers(self, field=0):
        """Device pointers of the two alternating trace buffers and of the half-step buffer of a wavefield."""
        b, n = (_vp * 3)(), _sz()
        self._ck(_lib.dg_get_trace_buffers(self._h, int(field), b, C.byref(n)))
        return [b[0], b[1], b[2]]

    def dg_halo_sources(self, src_trace_device):
        """Fused exchange: device pointers of the source buffer of every halo set, for the next (fine) step."""
        n = len(src_trace_device)
        arr = (_vp * max(n, 1))(*[_vp(int(x)) for x in src_trace_device])
        self._ck(_lib.dg_halo_sources(self._h, n, arr))

    # ---- RTM
    def rtm_set_receiver_capacity(self, max_receivers):
        self._ck(_lib.rtm_set_receiver_capacity(self._h, int(max_receivers)))

    def rtm_spill_bytes(self, nsteps):
        n = _sz()
        self._ck(_lib.rtm_spill_bytes(self._h, int(nsteps), C.byref(n)))
        return n.value

    def rtm_set_trace_spill(self, host_ptr, nbytes, window):
        self._ck(_lib.rtm_set_trace_spill(self._h, _vp(host_ptr), nbytes, int(window)))

    def rtm_set_spill_packing(self, on):
        self._ck(_lib.rtm_set_spill_packing(self._h, int(bool(on))))

    def spill_traces_torch(self, nsteps, window):
        """Pinned host tensor for the whole trace history; the RTM region bound afterwards keeps a ring of `window`."""
        import torch
        n = self.rtm_spill_bytes(nsteps)
        self._spill = torch.empty(n + 64, dtype=torch.uint8, pin_memory=True)
        base = (self._spill.data_ptr() + 15) & ~15
        self.rtm_set_trace_spill(base, n, window)
        return n

    def rtm_history_bytes(self, nsteps):
        n = _sz()
        self._ck(_lib.rtm_history_bytes(self._h, int(nsteps), C.byref(n)))
        return n.value

    def rtm_bind_history(self, dptr, nbytes):
        self._ck(_lib.rtm_bind_history(self._h, _vp(dptr), nbytes))

    def bind_history_torch(self, nsteps, device="cuda:0"):
        import torch
        n = self.rtm_history_bytes(nsteps)
        self._hist = torch.empty(n + 256, dtype=torch.uint8, device=device)
        base = (self._hist.data_ptr() + 255) & ~255
        self.rtm_bind_history(base, n)
        return n

    def rtm_forward_shot(self, nsteps, want_data=True):
        nloc = self.dg_get_dt()[1]
        data = np.empty((self.nr, nsteps * nloc + 1)) if (want_data and self.nr) else None
        self._ck(_lib.rtm_forward_shot(self._h, int(nsteps), _ptr(data, _pd)))
        return data

    def rtm_backward_shot(self, nsteps, data, updir=(0.0, 0.0, -1.0), imaging=DG_IMAGING_CHARACTERISTIC,
                          first_image_step=0):
        d = None if data is None else _f64(data)
        u = _f64(updir)
        self._ck(_lib.rtm_backward_shot(self._h, int(nsteps), _ptr(d, _pd), _ptr(u, _pd), int(imaging),
                                        int(first_image_step)))

    def rtm_forward_part(self, nsteps, fine0, nfine, want_data=True):
        """Fine steps [fine0, fine0 + nfine) of the forward phase; the recorded signals come back with the last part."""
        nloc = self.dg_get_dt()[1]
        last = fine0 + nfine == nsteps * nloc
        data = np.empty((self.nr, nsteps * nloc + 1)) if (want_data and self.nr and last) else None
        self._ck(_lib.rtm_forward_part(self._h, int(nsteps), int(fine0), int(nfine), _ptr(data, _pd)))
        return data

    def rtm_backward_part(self, nsteps, data, fine0, nfine, updir=(0.0, 0.0, -1.0), imaging=DG_IMAGING_CHARACTERISTIC,
                          first_image_step=0):
        d = None if data is None else _f64(data)
        u = _f64(updir)
        self._ck(_lib.rtm_backward_part(self._h, int(nsteps), _ptr(d, _pd), _ptr(u, _pd), int(imaging),
                                        int(first_image_step), int(fine0), int(nfine)))

    def rtm_get_trace_levels(self, field):
        L = int(self.dg_get_dt()[1]).bit_length()
        cur, half, n = (_vp * 8)(), _vp(), _sz()
        self._ck(_lib.rtm_get_trace_levels(self._h, int(field), cur, C.byref(half), C.byref(n)))
        return [cur[l] for l in range(L)], half.value, n.value

    def rtm_halo_sources(self, src_trace_device):
        n = len(src_trace_device)
        arr = (_vp * max(n, 1))(*[_vp(int(x)) for x in src_trace_device])
        self._ck(_lib.rtm_halo_sources(self._h, n, arr))

    def rtm_image_read(self):
        out = np.empty((self.K, self.Np))
        self._ck(_lib.rtm_image_read(self._h, _ptr(out, _pd)))
        return out

    def rtm_image_zero(self):
        self._ck(_lib.rtm_image_zero(self._h))

    def rtm_image_device(self):
        """(device pointer, bytes) of the image in the blocked device layout."""
        p, n = _vp(), _sz()
        self._ck(_lib.rtm_image_device(self._h, C.byref(p), C.byref(n)))
        return p.value, n.value

    def image_torch(self):
        """The device image as a 1-D torch view (float32 / float64) of the bound history tensor, for in-place
        collectives across replicas (argument marshalling only: no arithmetic happens here)."""
        import torch
        p, n = self.rtm_image_device()
        off = p - self._hist.data_ptr()
        assert 0 <= off and off + n <= self._hist.numel()
        return self._hist[off:off + n].view(torch.float64 if self.precision == 64 else torch.float32)

    # ---- getters
    def dg_get_nodes(self):
        r, s, t = (np.empty(self.Np) for _ in range(3))
        self._ck(_lib.dg_get_nodes(self._h, _ptr(r, _pd), _ptr(s, _pd), _ptr(t, _pd)))
        return r, s, t

    def dg_get_operators(self):
        Np, Nfp = self.Np, self.Nfp
        Dr, Ds, Dt = (np.empty((Np, Np)) for _ in range(3))
        LIFT = np.empty((Np, 4 * Nfp))
        Fmask = np.empty((4, Nfp), dtype=np.int32)
        self._ck(_lib.dg_get_operators(self._h, _ptr(Dr, _pd), _ptr(Ds, _pd), _ptr(Dt, _pd), _ptr(LIFT, _pd),
                                       _ptr(Fmask, _pi32)))
        return Dr, Ds, Dt, LIFT, Fmask

    def dg_get_connectivity(self):
        EToE = np.empty((self.K, 4), dtype=np.int32)
        EToF = np.empty((self.K, 4), dtype=np.int32)
        mapP = np.empty((self.K, 4, self.Nfp), dtype=np.int32)
        self._ck(_lib.dg_get_connectivity(self._h, _ptr(EToE, _pi32), _ptr(EToF, _pi32), _ptr(mapP, _pi32)))
        return EToE, EToF, mapP

    def dg_get_boundary_faces(self):
        bk, bf, bc = (np.empty(self.nbnd, dtype=np.int32) for _ in range(3))
        self._ck(_lib.dg_get_boundary_faces(self._h, _ptr(bk, _pi32), _ptr(bf, _pi32), _ptr(bc, _pi32)))
        return bk, bf, bc

    def dg_get_geometry(self):
        K = self.K
        J, ginv, nrm, gsur, ell = np.empty(K), np.empty((K, 3, 3)), np.empty((K, 4, 3)), np.empty((K, 4)), np.empty(K)
        self._ck(_lib.dg_get_geometry(self._h, _ptr(J, _pd), _ptr(ginv, _pd), _ptr(nrm, _pd), _ptr(gsur, _pd),
                                      _ptr(ell, _pd)))
        return dict(J=J, ginv=ginv, normals=nrm, gsur=gsur, ell=ell)

    def dg_get_levels(self):
        lv = np.empty(self.K, dtype=np.int32)
        self._ck(_lib.dg_get_levels(self._h, _ptr(lv, _pi32)))
        return lv

    def dg_get_dt(self):
        dt, nl = _d(), _i()
        self._ck(_lib.dg_get_dt(self._h, C.byref(dt), C.byref(nl)))
        return dt.value, nl.value

    def dg_get_time(self):
        t = _d()
        self._ck(_lib.dg_get_time(self._h, C.byref(t)))
        return t.value

    def dg_get_source(self):
        k = C.c_int32()
        w = np.empty(self.Np)
        self._ck(_lib.dg_get_source(self._h, C.byref(k), _ptr(w, _pd)))
        return k.value, w

    def dg_get_receivers(self):
        k = np.empty(self.nr, dtype=np.int32)
        rows, w = np.empty((self.nr, self.Np)), np.empty((self.nr, self.Np))
        self._ck(_lib.dg_get_receivers(self._h, _ptr(k, _pi32), _ptr(rows, _pd), _ptr(w, _pd)))
        return k, rows, w

    def dg_get_fields(self, out=None):
        """q[K][4][Np] in user order; `out` = a C-contiguous float64 array of that shape to fill instead of a new one."""
        q = np.empty((self.K, 4, self.Np)) if out is None else out
        assert q.shape == (self.K, 4, self.Np) and q.dtype == np.float64 and q.flags.c_contiguous
        self._ck(_lib.dg_get_fields(self._h, _ptr(q, _pd)))
        return q

    def dg_get_traces(self):
        qf = np.empty((self.K, 4, self.Nfp, 2))
        self._ck(_lib.dg_get_traces(self._h, _ptr(qf, _pd)))
        return qf

    def dg_get_rhs(self, which=DG_RHS_TOTAL, direction=1):
        r = np.empty((self.K, 4, self.Np))
        self._ck(_lib.dg_get_rhs(self._h, int(which), int(direction), _ptr(r, _pd)))
        return r

    def rtm_get_trace_index(self, level):
        nf, nrec = _i64(), _i64()
        self._ck(_lib.rtm_get_trace_index(self._h, int(level), C.byref(nf), C.byref(nrec), None))
        faces = np.empty(nf.value, dtype=np.int32)
        self._ck(_lib.rtm_get_trace_index(self._h, int(level), C.byref(nf), C.byref(nrec), _ptr(faces, _pi32)))
        return faces, nrec.value

    def rtm_get_traces(self, level, record):
        nf = self.rtm_get_trace_index(level)[0].size
        buf = np.empty((nf, self.Nfp, 2))
        self._ck(_lib.rtm_get_traces(self._h, int(level), int(record), _ptr(buf, _pd)))
        return buf

    def rtm_get_fields(self, which):
        q = np.empty((self.K, 4, self.Np))
        self._ck(_lib.rtm_get_fields(self._h, int(which), _ptr(q, _pd)))
        return q

    def dg_get_launch_count(self):
        n = _i64()
        self._ck(_lib.dg_get_launch_count(self._h, C.byref(n)))
        return n.value

    def dg_set_profiling(self, on):
        self._ck(_lib.dg_set_profiling(self._h, int(bool(on))))

    def dg_get_kernel_times(self):
        """{kernel class name: (milliseconds, launches)} since the last call (profiling mode)."""
        ms = np.zeros(len(KERNEL_CLASSES))
        cnt = np.zeros(len(KERNEL_CLASSES), dtype=np.int64)
        self._ck(_lib.dg_get_kernel_times(self._h, _ptr(ms, _pd), _ptr(cnt, _pi64)))
        return {n: (float(ms[i]), int(cnt[i])) for i, n in enumerate(KERNEL_CLASSES)}

    def dg_bench_kernel(self, which, reps):
        self._ck(_lib.dg_bench_kernel(self._h, int(which), int(reps)))


def dg_measure_fma(kind, device="cuda:0"):
    """TFLOP/s of a register-only FMA loop (kind 0 fp32 FFMA, 1 packed FFMA2, 2 fp64 DFMA)."""
    import torch
    buf = torch.empty(4 * 2048 * 256, dtype=torch.uint8, device=device)
    out = _d()
    with torch.cuda.device(device):
        rc = _lib.dg_measure_fma(int(kind), _vp(buf.data_ptr()), buf.numel(), _vp(torch.cuda.current_stream(device).cuda_stream),
                                 C.byref(out))
    if rc != DG_OK:
        raise DGError(rc, "dg_measure_fma")
    return out.value


def dg_version():
    return _lib.dg_version().decode()
