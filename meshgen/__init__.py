"""Seeded synthetic tetrahedral-mesh generators (inputs only).

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2106_01326_b200/``).  It holds none of the method's arithmetic: no
point-in-tetrahedron test, no bounding-box iteration, no voxel grid.  It only
builds ``verts int32[V][3]`` / ``tets int32[T][4]`` arrays from a seed.

The meshes stand in for the paper's Thingi10k / ModelNet tet meshes
(PAPER.md:28, :102-108, :273), which are not available; the recipe is stated in
DESIGN.md ("Input recipe").
"""
from .kuhn import (  # noqa: F401
    E_LATTICE,
    Mesh,
    kuhn_mesh,
    make_config,
    config_names,
    carve_every_third,
    carve_sphere,
    single_tet_mesh,
    lattice_form,
)
