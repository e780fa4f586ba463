"""Seeded synthetic INPUT generators shared by the oracle tests, the GPU tests and bench.py.

This package holds none of the method's arithmetic (no DG operators, no geometry factors, no
time stepping): it only produces plain arrays - tetrahedral meshes (EToV, VX), per-element
material (rho, c), source / receiver positions and the run parameters of the BASELINE.json
configurations.  Neither `oracle/` nor `paper_1506_00907_b200/` is imported from here.
"""
from .mesh import box_tet_mesh, permute_elements, graded_box_tet_mesh, box_side_bc  # noqa: F401
from .models import (two_layer_model, smooth_random_field, centroid_of_elements,  # noqa: F401
                     planted_reflector_model)
from .configs import make_config, CONFIG_NAMES  # noqa: F401
from .gathers import synthetic_gather  # noqa: F401
