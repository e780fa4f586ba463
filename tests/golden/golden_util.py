"""Compact summaries of a nodal array for stored expected values (test infrastructure).

A stored golden holds, per array x[K, ...]: the per-element Euclidean norms (float32, used as denominators only), M
seeded random projections per element (float64: any error in an element moves them; E|R^T e|^2 = M |e|^2 for standard
normal R) and the full values of a seeded element subset.  `compare` turns a candidate array into the same summary
and returns (estimated global relative L2 error, exact relative L2 error on the subset, largest per-element error
estimate relative to max(element norm, rms element norm))."""
import numpy as np

M_PROJ = 2


def _flat(x):
    x = np.asarray(x, dtype=np.float64)
    return x.reshape(x.shape[0], -1)


def _proj_matrix(width, seed):
    return np.random.default_rng(seed).standard_normal((width, M_PROJ))


def summarise(x, subset, seed):
    f = _flat(x)
    return dict(norm=np.linalg.norm(f, axis=1).astype(np.float32), proj=f @ _proj_matrix(f.shape[1], seed),
                sub=np.asarray(x, dtype=np.float64)[subset], subset=np.asarray(subset, dtype=np.int64),
                seed=np.int64(seed))


def pack(out, prefix, summary):
    for k, v in summary.items():
        out[prefix + "." + k] = v


def unpack(npz, prefix):
    return {k: npz[prefix + "." + k] for k in ("norm", "proj", "sub", "subset", "seed")}


def compare(x, gold):
    f = _flat(x)
    d = f @ _proj_matrix(f.shape[1], int(gold["seed"])) - gold["proj"]
    norm = gold["norm"].astype(np.float64)
    total = np.sqrt(np.sum(norm ** 2))
    est_global = np.sqrt(np.sum(d ** 2) / M_PROJ) / total
    sub = np.asarray(x, dtype=np.float64)[gold["subset"]]
    exact_subset = np.linalg.norm((sub - gold["sub"]).ravel()) / max(np.linalg.norm(gold["sub"].ravel()), 1e-300)
    rms = total / np.sqrt(len(norm))
    per_elem = np.sqrt(np.sum(d ** 2, axis=1) / M_PROJ) / np.maximum(norm, rms)
    return est_global, exact_subset, per_elem.max()
