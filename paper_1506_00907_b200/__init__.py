"""B200-native nodal DGTD / RTM hot path (arXiv 1506.00907) behind the C ABI of include/dgrtm.h.

    from paper_1506_00907_b200 import DG          # ctypes binding of libdgrtm.so (built in-tree)
    from paper_1506_00907_b200.decomp import Decomposition, partition_elements   # sub-domains with device halo exchange

`python -m paper_1506_00907_b200.build` compiles the library for sm_100a.  The binding is imported
lazily so that the build module can be run before the library exists; using any binding name without
the library raises ImportError (there is no CPU fallback).
"""
import importlib


def __getattr__(name):
    if name.startswith("__") or name in ("binding", "build", "decomp"):
        raise AttributeError(name)
    binding = importlib.import_module(__name__ + ".binding")
    if hasattr(binding, name):
        return getattr(binding, name)
    raise AttributeError("module %r has no attribute %r" % (__name__, name))
