"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no energies, no solver):
only mesh construction (icospheres mapped to cell rest shapes), the paper's
material table, and seeded random populations / forces shaped like the
paper's hematocrit workloads (Table 1).
Both `oracle/` and `paper_1911_03062_b200/` consumers receive the SAME arrays.
"""
from .meshes import (  # noqa: F401
    CellType,
    Material,
    icosahedron,
    icosphere,
    octasphere,
    rbc_material,
    platelet_material,
    rbc_cell_type,
    platelet_cell_type,
    icosahedron_cell_type,
)
from .populations import Population, make_config, CONFIG_NAMES  # noqa: F401
