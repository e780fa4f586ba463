"""dg_step_lserk4_static (include/dgrtm.h): the allocation-free variant of the LSERK4 time loop - the stage kernel's
2N-storage residual in a file-scope device array of the library (8 MiB, shared by every call on the GPU) instead of the
workspace.  Its output is compared with the existing path's (dg_step under DG_INTEGRATOR_LSERK4) on two calls in a row, with
a context of another order and precision using the shared array in between, and oversized states must be rejected.

Collected last on purpose (pytest -x): a failure here hides no other test."""
import numpy as np
import pytest

from workloads import make_config
from parity_util import make_gpu, rel_l2, random_state

pytestmark = pytest.mark.gpu

TOL = {64: 1e-10, 32: 1e-5}


def _pair(cfg, precision, q0):
    import paper_1506_00907_b200 as pk
    a, b = make_gpu(cfg, precision), make_gpu(cfg, precision)
    for g in (a, b):
        g.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
        g.dg_set_state(q0)
    return a, b


@pytest.mark.parametrize("name,N,precision", [("cfg1_cavity", 2, 64), ("cfg2_two_layer", 3, 32)])
def test_static_scratch_path_equals_the_workspace_path_on_two_calls(name, N, precision):
    import paper_1506_00907_b200 as pk
    assert pk.dg_static_scratch_bytes() == 8 << 20
    if name == "cfg1_cavity":
        cfg = make_config(name)                                       # BASELINE.json config 1: 384 tets, rigid walls, LSERK4
    else:
        cfg = make_config(name, hexes=(7, 6, 5), N=N)                 # 1 260 tets, point source, absorbing
        cfg["source"] = dict(cfg["source"], f0=40.0, tp=0.01)
    K, Np = cfg["EToV"].shape[0], (N + 1) * (N + 2) * (N + 3) // 6
    q0 = 1e-2 * random_state(K, Np, 5)
    old, new = _pair(cfg, precision, q0)
    # a context of another order / precision that dirties the shared array between the calls
    other_cfg = make_config("cfg2_two_layer", hexes=(4, 3, 3), N=4)
    other = make_gpu(other_cfg, 64 if precision == 32 else 32)
    other.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
    other.dg_set_state(1e3 * random_state(other.K, other.Np, 6))
    nsteps = 25
    for call in range(2):
        old.dg_step(nsteps)
        new.dg_step_lserk4_static(nsteps)
        qa, qb = old.dg_get_fields(), new.dg_get_fields()
        assert np.linalg.norm(qa) > 0 and np.isfinite(qb).all()
        assert rel_l2(qb, qa) < TOL[precision], (call, rel_l2(qb, qa))
        assert rel_l2(new.dg_get_traces(), old.dg_get_traces()) < TOL[precision]
        assert abs(new.dg_get_time() - old.dg_get_time()) < 1e-14
        other.dg_step_lserk4_static(3)                                # leaves its residual in the array
    for g in (old, new, other):
        g.close()


def test_static_scratch_rejects_states_beyond_its_size_and_wrong_modes():
    import paper_1506_00907_b200 as pk
    cfg = make_config("cfg2_two_layer", hexes=(16, 16, 12), N=4)      # 18 432 tets x 4 x 35 x 8 B = 20.6 MB > 8 MiB
    g = make_gpu(cfg, 64)
    g.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
    with pytest.raises(pk.DGError) as e:
        g.dg_step_lserk4_static(1)
    assert e.value.code == pk.DG_ERR_NOMEM and "8 MiB" in str(e.value)
    g.dg_step(1)                                                      # the workspace path still serves it
    g.close()
    small = make_gpu(make_config("cfg1_cavity"), 64)
    with pytest.raises(pk.DGError) as e:                              # AB3 is the default integrator
        small.dg_step_lserk4_static(1)
    assert e.value.code == pk.DG_ERR_STATE
    small.dg_set_integrator(pk.DG_INTEGRATOR_LSERK4)
    small.dg_set_profiling(True)
    with pytest.raises(pk.DGError):                                   # profiling creates events per launch
        small.dg_step_lserk4_static(1)
    small.dg_set_profiling(False)
    small.dg_step_lserk4_static(1)
    small.close()
