"""Boundary-trace spill to host memory (rtm_set_trace_spill): with a device ring
of a few records and the whole history in pinned host memory, the forward capture, the backward replay and the image are
BIT-identical to the run that keeps the history in HBM (the same kernels read the same values from another address), the
host copy equals the in-HBM records, and a second backward pass (which must fetch the late records again) reproduces the
first."""
import numpy as np
import pytest

from workloads import make_config
from parity_util import make_gpu

pytestmark = pytest.mark.gpu


def _shot(cfg, precision, nsteps, xr, spill_window, packed=False):
    import paper_1506_00907_b200 as pk
    g = pk.DG(cfg["N"], precision, cfg["EToV"], cfg["VX"], default_bc=cfg["default_bc"])
    g.dg_set_model(cfg["rho"], cfg["c"], cfg["nlevels"], cfg["cfl"])
    s = cfg["source"]
    g.dg_set_source(s["x0"], 40.0, 0.01, s["amp"])
    g.dg_set_receivers(xr)
    g.bind_torch("cuda:0")
    host_bytes = 0
    if spill_window:
        if packed:
            g.rtm_set_spill_packing(True)
        host_bytes = g.spill_traces_torch(nsteps, spill_window)
    nb = g.bind_history_torch(nsteps, "cuda:0")
    data = g.rtm_forward_shot(nsteps)
    qT = g.rtm_get_fields(0)
    recs = {}
    for lev in range(cfg["nlevels"]):
        faces, nrec = g.rtm_get_trace_index(lev)
        if len(faces):
            recs[lev] = [g.rtm_get_traces(lev, j) for j in (0, 1, nrec // 2, nrec - 2, nrec - 1)]
    g.rtm_backward_shot(nsteps, data, updir=(0.0, 0.0, -1.0))
    img1 = g.rtm_image_read()
    fs = g.rtm_get_fields(1)
    g.rtm_image_zero()
    g.rtm_backward_shot(nsteps, data, updir=(0.0, 0.0, -1.0))      # the ring now holds early records: fetch again
    img2 = g.rtm_image_read()
    g.close()
    return dict(data=data, qT=qT, recs=recs, img1=img1, img2=img2, fs=fs, hist_bytes=nb, host_bytes=host_bytes)


@pytest.mark.parametrize("name,N,precision,window", [("cfg2_two_layer", 3, 32, 4), ("cfg3_lts", 3, 32, 3),
                                                     ("cfg3_lts", 2, 64, 2), ("cfg2_two_layer", 4, 32, 8)])
def test_spilled_history_is_bit_identical(name, N, precision, window):
    hexes = (6, 6, 8) if name == "cfg3_lts" else (7, 6, 5)
    nsteps = 40
    cfg = make_config(name, hexes=hexes, N=N, nsteps=nsteps)
    gx = np.linspace(0.4, 2.6, 3)
    xr = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
    a = _shot(cfg, precision, nsteps, xr, 0)
    b = _shot(cfg, precision, nsteps, xr, window)
    assert b["hist_bytes"] < a["hist_bytes"]                       # the device keeps a ring only
    assert np.array_equal(a["data"], b["data"]) and np.array_equal(a["qT"], b["qT"])
    assert a["recs"].keys() == b["recs"].keys() and len(a["recs"]) > 0
    for lev in a["recs"]:
        for ra, rb in zip(a["recs"][lev], b["recs"][lev]):
            assert np.array_equal(ra, rb) and np.abs(ra).max() >= 0
    assert np.abs(a["img1"]).max() > 0
    assert np.array_equal(a["img1"], b["img1"]) and np.array_equal(a["fs"], b["fs"])
    assert np.array_equal(b["img1"], b["img2"]) and np.array_equal(a["img1"], a["img2"])


@pytest.mark.parametrize("name,N,precision,window", [("cfg2_two_layer", 3, 64, 4), ("cfg3_lts", 3, 32, 3)])
def test_packed_host_copy_halves_the_bytes_within_its_rounding(name, N, precision, window):
    """rtm_set_spill_packing: the host copy of the history in half the bytes (fp64 -> fp32, fp32 -> bf16).  Lossy by design:
    the forward phase is untouched (bit-identical data and final state), every stored value comes back within the storage
    format's rounding (2^-24 / 2^-8 relative), and the reconstructed source field and the image move by that order."""
    hexes = (6, 6, 8) if name == "cfg3_lts" else (7, 6, 5)
    nsteps = 40
    cfg = make_config(name, hexes=hexes, N=N, nsteps=nsteps)
    gx = np.linspace(0.4, 2.6, 3)
    xr = np.array([[x + 0.013, y + 0.007, 0.06] for x in gx for y in gx])
    a = _shot(cfg, precision, nsteps, xr, window)                     # lossless spill
    b = _shot(cfg, precision, nsteps, xr, window, packed=True)
    assert 0 < b["host_bytes"] <= a["host_bytes"] // 2 + 256 * cfg["nlevels"]
    assert np.array_equal(a["data"], b["data"]) and np.array_equal(a["qT"], b["qT"])
    eps = 2.0 ** -24 if precision == 64 else 2.0 ** -8
    for lev in a["recs"]:
        for ra, rb in zip(a["recs"][lev], b["recs"][lev]):
            assert np.abs(ra - rb).max() <= eps * np.abs(ra).max() * 1.001 + 1e-300
    rel = lambda x, y: np.linalg.norm((x - y).ravel()) / np.linalg.norm(y.ravel())
    assert np.abs(a["img1"]).max() > 0
    err_f, err_i = rel(b["fs"], a["fs"]), rel(b["img1"], a["img1"])
    assert err_f < 20 * eps and err_i < 20 * eps, (err_f, err_i)
    assert err_i > 0                                                  # it IS lossy: the packing was in the path
    assert np.array_equal(b["img1"], b["img2"])                       # deterministic: the second pass fetches the same values
