"""CPU-only checks of the boundary: libdgrtm.so builds in-tree, loads, exports every symbol that
include/dgrtm.h declares, and the host-only calls (no device) behave as the header states."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from workloads import box_tet_mesh

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1506_00907_b200.build import build
    return build()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "dgrtm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b((?:dg|rtm)_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib_path):
    names = _declared_functions()
    assert len(names) >= 35
    lib = C.CDLL(lib_path)
    for n in names:
        assert hasattr(lib, n), "libdgrtm.so does not export %s" % n
    from paper_1506_00907_b200 import binding
    assert sorted(binding.SIGNATURES) == names, "binding and header disagree"


def test_host_only_calls(lib_path):
    """Setup runs on the host: mesh, model, levels, sizes, error codes - no device needed."""
    import paper_1506_00907_b200 as pk
    assert "sm_100a" in pk.dg_version()
    etov, vx = box_tet_mesh(2, 2, 2, jitter=0.1, seed=1)
    g = pk.DG(3, 32, etov, vx)
    assert (g.K, g.Np, g.Nfp, g.nbnd) == (48, 20, 10, 48)
    with pytest.raises(pk.DGError) as e:
        g.dg_workspace_bytes()
    assert e.value.code == pk.DG_ERR_STATE
    g.dg_set_model(np.ones(48), np.ones(48), 2, 0.15)
    assert g.dg_workspace_bytes() > 48 * 4 * 20 * 4 * 4
    assert g.rtm_history_bytes(10) > 0
    n0 = g.rtm_history_bytes(10)
    g.rtm_set_receiver_capacity(1000)                       # sizes the receiver-dependent part of the RTM region
    assert g.rtm_history_bytes(10) > n0 + 1000 * 11 * 4
    g.rtm_set_receiver_capacity(0)
    assert g.rtm_history_bytes(10) == n0
    dt, nloc = g.dg_get_dt()
    assert dt > 0 and nloc == 2
    lv = g.dg_get_levels()
    assert lv.min() >= 0 and lv.max() <= 1
    with pytest.raises(pk.DGError) as e:
        g.dg_step(1)
    assert e.value.code == pk.DG_ERR_STATE
    bad = etov.copy()
    bad[0, [0, 1]] = bad[0, [1, 0]]
    with pytest.raises(pk.DGError) as e:
        pk.DG(3, 32, bad, vx)
    assert e.value.code == pk.DG_ERR_MESH
    g.close()


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may import it (or workloads')
    arithmetic, and the oracle imports nothing of the package."""
    pkg = os.path.join(ROOT, "paper_1506_00907_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "oracle/" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1506_00907_b200" not in s.replace("(paper_1506_00907_b200/)", ""), f
