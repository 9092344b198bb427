"""B200-native tetrahedral-mesh -> solid-binary-voxel hot path (arxiv 2106.01326).

Thin Python binding over the C-ABI library ``libvox.so`` (``include/vox.h``):
argument marshalling only -- every step of the path runs in the CUDA kernels of
``csrc/vox.cu``.  There is no CPU fallback: importing works without a GPU (so
that the build can be checked), but every compute call needs the library and a
CUDA device and fails loudly otherwise.
"""
from .binding import (  # noqa: F401
    Pipe,
    VoxError,
    Voxelizer,
    debug_check_status,
    kernel_launches,
    lib_path,
    load_library,
    occupancy,
    probe_int32,
    voxelize,
    voxelize_host,
    EXPORTS,
)
