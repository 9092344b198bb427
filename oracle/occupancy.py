"""Oracle for the sub-sample occupancy count.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Definition (include/vox.h "Occupancy from sub-samples"; the paper only says each model is "voxelized into 5
million samples, with a resolution of 256^3"): voxel (x,y,z) of the coarse grid owns the k^3
voxel centres (k*x+i, k*y+j, k*z+l), 0 <= i,j,l < k, of the grid k times finer per axis; its count is the
number of those fine samples that are solid.  Written out with numpy on the unpacked fine bit grid; shares
nothing with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def occupancy(dense_fine: np.ndarray, k: int) -> np.ndarray:
    """dense_fine uint32[batch][k*nz][k*ny][k*nx/32] (LSB = lowest x) -> uint8[batch][nz][ny][nx]."""
    b, fz, fy, fw = dense_fine.shape
    bits = np.unpackbits(np.ascontiguousarray(dense_fine).view(np.uint8).reshape(b, fz, fy, fw * 4),
                         axis=-1, bitorder="little")          # [b][fz][fy][fx], x ascending
    fx = fw * 32
    assert fz % k == 0 and fy % k == 0 and fx % k == 0
    v = bits.reshape(b, fz // k, k, fy // k, k, fx // k, k).astype(np.uint16)
    return v.sum(axis=(2, 4, 6)).astype(np.uint8)
