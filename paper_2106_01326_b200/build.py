"""Build the C-ABI library ``libvox.so`` in-tree with nvcc for sm_100a.

``python -m paper_2106_01326_b200.build`` or ``build()``; cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "vox.cu")  # the one translation unit; it includes the .cuh parts beside it
HDR = os.path.join(os.path.dirname(_HERE), "include", "vox.h")


def _deps():
    d = os.path.dirname(SRC)
    return [os.path.join(d, f) for f in sorted(os.listdir(d)) if f.endswith((".cu", ".cuh", ".h"))] + [HDR]
LIB = os.path.join(_HERE, "libvox.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


LIB_CHECKED = os.path.join(_HERE, "libvox_checked.so")


def build_checked(force: bool = False) -> str:
    """The same source with -DVOX_CHECKS: device-side bounds checks on every index the kernels form
    (vox_debug_check_status; tests/test_gpu_checked_build.py)."""
    if force or not os.path.exists(LIB_CHECKED) or any(
            os.path.getmtime(f) > os.path.getmtime(LIB_CHECKED) for f in _deps()):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB_CHECKED + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc] + NVCC_FLAGS + ["-DVOX_CHECKS", "-o", tmp, SRC])
        os.replace(tmp, LIB_CHECKED)
    return LIB_CHECKED


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    m = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > m for f in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
