"""ctypes loader for ``voxel_oracle.c`` (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Builds ``liboracle.so`` beside the source with gcc on first use.  Holds no
arithmetic of its own: argument marshalling only.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "voxel_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile voxel_oracle.c -> liboracle.so (gcc -O2 -fopenmp).  Returns the path."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            subprocess.check_call(
                ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC]
            )
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i32p = ctypes.POINTER(ctypes.c_int32)
        i64p = ctypes.POINTER(ctypes.c_int64)
        lib.oracle_voxelize.restype = ctypes.c_int
        lib.oracle_voxelize.argtypes = [
            i32p, ctypes.c_int64, i32p, ctypes.c_int64, i64p, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_int, ctypes.c_int64, ctypes.POINTER(ctypes.c_uint32), i64p,
        ]
        lib.oracle_determinants.restype = None
        lib.oracle_determinants.argtypes = [i32p, i32p, i32p, i32p, i32p, i64p]
        lib.oracle_inside.restype = ctypes.c_int
        lib.oracle_inside.argtypes = [i32p, i32p, i32p, i32p, i32p]
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def voxelize(verts, tets, grid, extent=(65536, 65536, 65536), tet_offsets=None, mode=0,
             tet_stride=1, return_samples=False):
    """Solid bit grid of a (batched) tet mesh.

    verts int32[V][3], tets int32[T][4]; grid=(nx,ny,nz); extent=(ex,ey,ez);
    tet_offsets int64[batch+1] or None.  Returns uint32[batch][nz][ny][nx/32]
    (and the candidate-sample count if asked).
    """
    lib = _load()
    verts = np.ascontiguousarray(verts, dtype=np.int32).reshape(-1, 3)
    tets = np.ascontiguousarray(tets, dtype=np.int32).reshape(-1, 4)
    nx, ny, nz = (int(g) for g in grid)
    ex, ey, ez = (int(e) for e in extent)
    if tet_offsets is None:
        tet_offsets = np.array([0, len(tets)], dtype=np.int64)
    tet_offsets = np.ascontiguousarray(tet_offsets, dtype=np.int64)
    batch = len(tet_offsets) - 1
    bits = np.empty((batch, nz, ny, nx // 32), dtype=np.uint32)
    samples = ctypes.c_int64(0)
    rc = lib.oracle_voxelize(
        _p(verts, ctypes.c_int32), len(verts), _p(tets, ctypes.c_int32), len(tets),
        _p(tet_offsets, ctypes.c_int64), batch, nx, ny, nz, ex, ey, ez, int(mode),
        int(tet_stride), _p(bits, ctypes.c_uint32), ctypes.byref(samples),
    )
    if rc != 0:
        raise ValueError("oracle_voxelize: invalid arguments")
    return (bits, int(samples.value)) if return_samples else bits


def determinants(P, A, B, C, D):
    """(Da, Db, Dc, Dd, 6V) of Theorem 1 for one point and one tet (int64)."""
    arrs = [np.ascontiguousarray(v, dtype=np.int32) for v in (P, A, B, C, D)]
    out = np.zeros(5, dtype=np.int64)
    _load().oracle_determinants(*[_p(a, ctypes.c_int32) for a in arrs], _p(out, ctypes.c_int64))
    return [int(v) for v in out]


def inside(P, A, B, C, D) -> bool:
    arrs = [np.ascontiguousarray(v, dtype=np.int32) for v in (P, A, B, C, D)]
    return bool(_load().oracle_inside(*[_p(a, ctypes.c_int32) for a in arrs]))
