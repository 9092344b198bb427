"""CPU oracle for the tet-mesh -> solid-voxel step.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2106_01326_b200`` and shares no code with the CUDA path.

Two independent implementations of the same plain definition (DESIGN.md
"Oracle"):

  * ``voxel_oracle.c``  -- plain C, int64_t, direct cofactor determinants per
    sample (``voxelize``);
  * ``bruteforce.py``   -- pure Python big integers, all voxels x all tets, no
    bounding box (tiny inputs; pins the C one).

plus the plain definitions of the two derived outputs: ``sparse.py`` (two-level tile encoding) and
``occupancy.py`` (k^3 sub-sample counts).
"""
from .binding import (  # noqa: F401
    build,
    determinants,
    inside,
    num_threads,
    voxelize,
)
from .bruteforce import bruteforce_voxelize, inside_closed_py  # noqa: F401
