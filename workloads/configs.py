"""The five BASELINE.json configurations as seeded synthetic inputs (recipe: DESIGN.md "Inputs").

`make_config(name, hexes=None, ...)` returns a dict of plain arrays / numbers:
  EToV, VX, rho, c, N, precision (32|64), default_bc, nlevels, cfl, integrator ("ab3"|"lserk4"),
  nsteps (global steps), lengths, source (x0, f0, tp, amp) or None, receivers [nr,3] or None,
  updir, c_true (config 4 only), initial ("cavity_mode"|"rest").
`hexes=(nx,ny,nz)` overrides the resolution (the parity tests use reduced meshes the oracle
finishes in seconds); everything else follows from the seed.
"""
import numpy as np

from .mesh import box_tet_mesh, graded_box_tet_mesh
from .models import (two_layer_model, smooth_random_field, planted_reflector_model)

BC_FREE, BC_ABSORBING, BC_RIGID, BC_PRESCRIBED = 1, 2, 3, 4
CONFIG_NAMES = ("cfg1_cavity", "cfg2_two_layer", "cfg3_lts", "cfg4_rtm", "cfg5_sweep")


def _source_top_centre(lengths, hexes):
    hx = lengths[0] / hexes[0]
    hz = lengths[2] / hexes[2]
    # top centre, a quarter cell below the surface, moved off the mesh planes
    return np.array([0.5 * lengths[0] + 0.013 * hx, 0.5 * lengths[1] + 0.007 * hx, 0.25 * hz])


def _receiver_grid(lengths, hexes, n_side):
    hz = lengths[2] / hexes[2]
    hx = lengths[0] / hexes[0]
    gx = np.linspace(0.1 * lengths[0], 0.9 * lengths[0], n_side) + 0.011 * hx
    gy = np.linspace(0.1 * lengths[1], 0.9 * lengths[1], n_side) + 0.017 * hx
    X, Y = np.meshgrid(gx, gy, indexing="ij")
    return np.stack([X.ravel(), Y.ravel(), np.full(X.size, 0.2 * hz)], axis=1)


def make_config(name, hexes=None, N=None, precision=None, nsteps=None, n_receivers_side=None):
    if name == "cfg1_cavity":
        hx = hexes or (4, 4, 4)
        lengths = (1.0, 1.0, 1.0)
        etov, vx = box_tet_mesh(*hx, lengths=lengths)
        K = etov.shape[0]
        cfg = dict(EToV=etov, VX=vx, rho=np.ones(K), c=np.ones(K), N=N or 2,
                   precision=precision or 64, default_bc=BC_RIGID, nlevels=1, cfl=0.5,
                   integrator="lserk4", nsteps=nsteps or 100, lengths=lengths, source=None,
                   receivers=None, initial="cavity_mode", seed=None)
    elif name == "cfg2_two_layer":
        hx = hexes or (32, 32, 16)
        lengths = (3.0, 3.0, 1.5)
        etov, vx = box_tet_mesh(*hx, lengths=lengths, jitter=0.1, seed=2)
        rho, c = two_layer_model(etov, vx, 0.75, 1.5, 1.0, 3.0, 2.2)
        cfg = dict(EToV=etov, VX=vx, rho=rho, c=c, N=N or 3, precision=precision or 32,
                   default_bc=BC_ABSORBING, nlevels=1, cfl=0.15, integrator="ab3",
                   nsteps=nsteps or 1000, lengths=lengths,
                   source=dict(x0=_source_top_centre(lengths, hx), f0=15.0, tp=0.1, amp=1.0),
                   receivers=None, initial="rest", seed=2)
    elif name == "cfg3_lts":
        hx = hexes or (48, 48, 24)
        lengths = (3.0, 3.0, 1.5)
        etov, vx = graded_box_tet_mesh(*hx, lengths=lengths, band_center=0.75, band_width=0.2,
                                       max_ratio=4.0, seed=3)
        c = smooth_random_field(etov, vx, lengths, 1.5, 4.5, seed=33)
        cfg = dict(EToV=etov, VX=vx, rho=np.ones(etov.shape[0]), c=c, N=N or 4,
                   precision=precision or 32, default_bc=BC_ABSORBING, nlevels=3, cfl=0.15,
                   integrator="ab3", nsteps=nsteps or 500, lengths=lengths,
                   source=dict(x0=_source_top_centre(lengths, hx), f0=15.0, tp=0.1, amp=1.0),
                   receivers=None, initial="rest", seed=3)
    elif name == "cfg4_rtm":
        hx = hexes or (64, 64, 32)
        lengths = (3.0, 3.0, 1.5)
        etov, vx = box_tet_mesh(*hx, lengths=lengths, jitter=0.1, seed=4)
        noise = smooth_random_field(etov, vx, lengths, 0.0, 1.0, seed=44)
        zc = vx[etov].mean(axis=1)[:, 2] / lengths[2]
        c = 1.5 + 2.0 * np.clip(0.6 * noise + 0.4 * zc, 0.0, 1.0)          # in [1.5, 3.5]
        hz = lengths[2] / hx[2]
        c_true = planted_reflector_model(etov, vx, lengths, c, depth0=3.7 * hz, dip_x=0.02,
                                         dip_y=-0.01, factor=1.3)
        cfg = dict(EToV=etov, VX=vx, rho=np.ones(etov.shape[0]), c=c, c_true=c_true, N=N or 3,
                   precision=precision or 32, default_bc=BC_ABSORBING, nlevels=1, cfl=0.15,
                   integrator="ab3", nsteps=nsteps or 2000, lengths=lengths,
                   source=dict(x0=_source_top_centre(lengths, hx), f0=15.0, tp=0.1, amp=1.0),
                   receivers=_receiver_grid(lengths, hx, n_receivers_side or 64),
                   updir=np.array([0.0, 0.0, -1.0]), initial="rest", seed=4)
    elif name == "cfg5_sweep":
        hx = hexes or (96, 96, 48)
        lengths = (3.0, 3.0, 1.5)
        etov, vx = graded_box_tet_mesh(*hx, lengths=lengths, band_center=0.75, band_width=0.2,
                                       max_ratio=4.0, seed=5)
        rng = np.random.default_rng(5)
        hxyz = np.array([lengths[0] / hx[0], lengths[1] / hx[1], 0.0])     # jitter x,y only
        inner = np.ones(vx.shape[0], dtype=bool)
        for d in range(3):
            inner &= (vx[:, d] > 1e-12) & (vx[:, d] < lengths[d] * (1 - 1e-12))
        vx = vx + rng.uniform(-0.1, 0.1, size=vx.shape) * hxyz * inner[:, None]
        rho = smooth_random_field(etov, vx, lengths, 1.0, 2.5, seed=55)
        c = smooth_random_field(etov, vx, lengths, 1.5, 4.5, seed=56)
        cfg = dict(EToV=etov, VX=vx, rho=rho, c=c, N=N or 3, precision=precision or 32,
                   default_bc=BC_ABSORBING, nlevels=3, cfl=0.15, integrator="ab3",
                   nsteps=nsteps or 200, lengths=lengths,
                   source=dict(x0=_source_top_centre(lengths, hx), f0=15.0, tp=0.1, amp=1.0),
                   receivers=None, initial="rest", seed=5)
    else:
        raise ValueError(f"unknown config {name!r}; one of {CONFIG_NAMES}")
    cfg["name"] = name
    cfg["hexes"] = tuple(hx)
    return cfg
