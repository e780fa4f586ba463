"""Writes the stored expected values tests/golden/*.npz of the GPU-filling, full-length parity tests
(tests/test_gpu_goldens.py).  Calls ONLY oracle/ (the fp64 numpy oracle of the paper's scheme) and workloads/ (seeded
inputs); nothing here touches the CUDA path.

    python tests/golden/make_goldens.py cfg2 cfg3 cfg4 bc        # any subset; minutes to hours of numpy each

Mesh of every case: 24 x 24 x 12 hexahedra x 6 = 41 472 tetrahedra = 1 296 blocks of 32 elements (about 3 work items
per group of the pipelined step kernel, ragged per-CTA chunks), the scaled mesh of SURVEY.md 8(d) "Oracle timing
beside it".
  cfg2: BASELINE.json config 2 at full length (N = 3, two layers, 15 Hz Ricker, absorbing, 1000 steps single rate);
  cfg3: config-3 shape (graded mesh, three multi-rate levels, N = 4), 100 global steps;
  cfg4: config-4 shape RTM shot, N = 3, 64 x 64 receivers, 2000 forward steps with trace capture and recording,
        2000 backward steps (trace replay, injection of a seeded synthetic gather, characteristic imaging (7));
  bc  : N = 3, one boundary type per box side (free-surface top, rigid bottom, absorbing sides), 300 steps.
Each array is stored as a summary (golden_util.summarise): per-element norms, seeded projections, and the full values
of a seeded element subset that contains boundary elements, level-interface elements and the point-term elements.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, HERE)

from golden_util import summarise, pack                      # noqa: E402
from oracle.dgtd import DGOracle                             # noqa: E402
from workloads import make_config, synthetic_gather, box_side_bc          # noqa: E402

HEXES = (24, 24, 12)


def build(cfg, face_bc=None):
    o = DGOracle(cfg["N"], cfg["EToV"], cfg["VX"], face_bc=face_bc, default_bc=cfg["default_bc"])
    o.set_model(cfg["rho"], cfg["c"], cfg["nlevels"], cfg["cfl"])
    if cfg.get("source"):
        s = cfg["source"]
        o.set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    if cfg.get("receivers") is not None:
        o.set_receivers(cfg["receivers"])
    return o


def element_subset(o, seed, n=192):
    """Seeded subset: random elements + boundary elements + elements at a level interface + point-term elements."""
    rng = np.random.default_rng(seed)
    K = o.K
    pick = [rng.choice(K, n // 2, replace=False)]
    bnd = np.nonzero((o.EToE < 0).any(axis=1))[0]
    pick.append(rng.choice(bnd, min(n // 4, bnd.size), replace=False))
    nb_level = np.where(o.EToE >= 0, o.level[np.maximum(o.EToE, 0)], o.level[:, None])
    iface = np.nonzero((nb_level != o.level[:, None]).any(axis=1))[0]
    if iface.size:
        pick.append(rng.choice(iface, min(n // 4, iface.size), replace=False))
    if o.source is not None:
        pick.append(np.array([o.source["k"]]))
    if o.receivers is not None:
        pick.append(o.receivers["k"][:: max(1, len(o.receivers["k"]) // 16)])
    return np.unique(np.concatenate(pick))


def make_cfg2(out):
    cfg = make_config("cfg2_two_layer", hexes=HEXES)
    o = build(cfg)
    F = o.new_field()
    o.run_mrab([F], cfg["nsteps"], 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    sub = element_subset(o, 20)
    pack(out, "q", summarise(F.q, sub, 201))
    out["nsteps"] = np.int64(cfg["nsteps"])
    out["dt_local"] = np.float64(o.dt_local)


def make_cfg3(out):
    cfg = make_config("cfg3_lts", hexes=HEXES, N=4, nsteps=100)
    o = build(cfg)
    assert len(np.unique(o.level)) == 3
    F = o.new_field()
    o.run_mrab([F], cfg["nsteps"], 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    sub = element_subset(o, 30)
    pack(out, "q", summarise(F.q, sub, 301))
    out["level_hist"] = np.bincount(o.level, minlength=3).astype(np.int64)
    out["nsteps"] = np.int64(cfg["nsteps"])
    out["dt_local"] = np.float64(o.dt_local)


def make_bc(out):
    cfg = make_config("cfg2_two_layer", hexes=HEXES, nsteps=300)
    cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)           # active within 300 steps, reaches the free surface
    o = build(cfg, face_bc=box_side_bc(cfg["EToV"], cfg["VX"], cfg["lengths"]))
    F = o.new_field()
    o.run_mrab([F], cfg["nsteps"], 0.0, 1, source_on=(True,))
    assert np.linalg.norm(F.q) > 0
    sub = element_subset(o, 40)
    pack(out, "q", summarise(F.q, sub, 401))
    out["bc_hist"] = np.bincount(o.bc[o.bnd_k, o.bnd_f], minlength=5).astype(np.int64)
    out["nsteps"] = np.int64(cfg["nsteps"])


def make_cfg4(out):
    cfg = make_config("cfg4_rtm", hexes=HEXES)
    nsteps = cfg["nsteps"]
    o = build(cfg)
    t0 = time.time()
    data, hist, qT = o.rtm_forward(nsteps)
    print("forward phase %.0f s" % (time.time() - t0), flush=True)
    sub = element_subset(o, 50)
    pack(out, "qT", summarise(qT, sub, 501))
    rng = np.random.default_rng(51)
    nr = data.shape[0]
    rsel = np.sort(rng.choice(nr, 64, replace=False))
    tsel = np.array([0, 1, nsteps // 4, nsteps // 2, nsteps - 1, nsteps], dtype=np.int64)
    out["data_rcv_sel"] = rsel
    out["data_rcv"] = data[rsel]                                    # full traces of 64 receivers
    out["data_t_sel"] = tsel
    out["data_t"] = data[:, tsel]                                   # all receivers at 6 sample times
    out["data_norm"] = np.float64(np.linalg.norm(data))
    faces = hist.faces[0]
    fsel = np.sort(rng.choice(faces.size, 256, replace=False))
    out["trace_faces"] = faces.astype(np.int64)                     # boundary-face-list indices (bit-exact)
    out["trace_face_sel"] = fsel
    out["trace_rec_sel"] = tsel
    out["trace_rec"] = hist.records[0][tsel][:, fsel]
    out["trace_max"] = np.float64(np.abs(hist.records[0]).max())
    # backward phase on a seeded synthetic gather (an input; see workloads/gathers.py)
    d = synthetic_gather(cfg["receivers"], cfg["source"]["x0"], nsteps + 1, o.dt_local, seed=52)
    t0 = time.time()
    I, FS, FR = o.rtm_backward(nsteps, qT, hist, d, updir=cfg["updir"], mode="characteristic", nglobal_total=nsteps)
    print("backward phase %.0f s" % (time.time() - t0), flush=True)
    assert np.abs(I).max() > 0
    pack(out, "FS", summarise(FS.q, sub, 502))
    pack(out, "FR", summarise(FR.q, sub, 503))
    pack(out, "I", summarise(I, sub, 504))
    out["nsteps"] = np.int64(nsteps)
    out["dt_local"] = np.float64(o.dt_local)
    out["gather_seed"] = np.int64(52)


CASES = dict(cfg2=make_cfg2, cfg3=make_cfg3, cfg4=make_cfg4, bc=make_bc)

if __name__ == "__main__":
    for name in sys.argv[1:] or list(CASES):
        t0 = time.time()
        out = {}
        CASES[name](out)
        path = os.path.join(HERE, "%s_24x24x12.npz" % name)
        np.savez(path, **out)
        print("%s: %.0f s -> %s (%.1f MB)" % (name, time.time() - t0, path, os.path.getsize(path) / 1e6), flush=True)
