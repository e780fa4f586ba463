"""Helpers of the parity tests: build the oracle and the CUDA path (through the C ABI) from the same
seeded inputs of `workloads`, and compare.  Holds none of the method's arithmetic."""
import numpy as np


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    nb = np.linalg.norm(b.ravel())
    return np.linalg.norm((a - b).ravel()) / (nb if nb > 0 else 1.0)


def make_oracle(cfg, nlevels=None, face_bc=None):
    from oracle.dgtd import DGOracle
    dg = DGOracle(cfg["N"], cfg["EToV"], cfg["VX"], face_bc=face_bc, default_bc=cfg["default_bc"])
    dg.set_model(cfg["rho"], cfg["c"], nlevels or cfg["nlevels"], cfg["cfl"])
    if cfg.get("source"):
        s = cfg["source"]
        dg.set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    if cfg.get("receivers") is not None:
        dg.set_receivers(cfg["receivers"])
    return dg


def make_gpu(cfg, precision=None, nlevels=None, face_bc=None, history_steps=None):
    """DG ctx of the CUDA path, workspace (and RTM history) bound to torch uint8 tensors."""
    import paper_1506_00907_b200 as pk
    g = pk.DG(cfg["N"], precision or cfg["precision"], cfg["EToV"], cfg["VX"], face_bc=face_bc,
              default_bc=cfg["default_bc"])
    g.dg_set_model(cfg["rho"], cfg["c"], nlevels or cfg["nlevels"], cfg["cfl"])
    if cfg.get("source"):
        s = cfg["source"]
        g.dg_set_source(s["x0"], s["f0"], s["tp"], s["amp"])
    if cfg.get("receivers") is not None:
        g.dg_set_receivers(cfg["receivers"])
    g.bind_torch()
    if history_steps:
        g.bind_history_torch(history_steps)
    return g


def cavity_mode(X, t, rho=1.0, c=1.0):
    """Closed-form rigid-wall cavity mode of the unit cube (SURVEY.md 8(c) pins), q[K,4,Np]."""
    w = np.sqrt(3.0) * np.pi * c
    cx, cy, cz = [np.cos(np.pi * X[..., d]) for d in range(3)]
    sx, sy, sz = [np.sin(np.pi * X[..., d]) for d in range(3)]
    q = np.zeros((X.shape[0], 4, X.shape[1]))
    q[:, 0] = cx * cy * cz * np.cos(w * t)
    a = np.pi / (rho * w) * np.sin(w * t)
    q[:, 1] = a * sx * cy * cz
    q[:, 2] = a * cx * sy * cz
    q[:, 3] = a * cx * cy * sz
    return q


def random_state(K, Np, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((K, 4, Np))
