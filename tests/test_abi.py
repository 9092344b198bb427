"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol
include/vox.h declares, and its host-only entry points validate their arguments.
No compute call is made (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2106_01326_b200.build import build

    build()
    import paper_2106_01326_b200 as pkg

    return pkg.load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "vox.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(vox_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    import paper_2106_01326_b200 as pkg

    names = _declared()
    assert len(names) >= 15
    assert sorted(pkg.EXPORTS) == names
    for n in names:
        assert getattr(lib, n) is not None


def test_header_is_plain_c():
    src = open(os.path.join(ROOT, "include", "vox.h")).read()
    assert 'extern "C"' in src and "torch" not in src.lower().replace("pytorch", "")


def test_create_validates(lib):
    c = ctypes.c_void_p()
    E = 65536
    ok = lib.vox_create(ctypes.byref(c), 1024, 1024, 1024, E, E, E, 1)
    assert ok == 0 and c.value
    assert lib.vox_grid_words(c) == 1024 * 1024 * 32
    assert lib.vox_workspace_fixed_bytes(c) > 0
    # order violation: vox_run before vox_tets
    assert lib.vox_run(c, None, ctypes.c_void_p(256), 1 << 20, ctypes.c_void_p(256)) == -5
    assert lib.vox_set_tile(c, 16, 8) == 0
    assert lib.vox_set_tile(c, 12, 8) == -1
    assert lib.vox_set_tile(c, 64, 8) == -1
    lib.vox_destroy(c)
    bad = [
        (100, 32, 32, E, E, E, 1),      # nx % 32
        (32, 32, 32, E + 2, E, E, 1),   # extent % 2n
        (32, 32, 48, E, E, E, 1),       # 65536 % 96
        (32, 32, 32, E, E, E, 0),       # batch
        (0, 32, 32, E, E, E, 1),
        (32, -1, 32, E, E, E, 1),
    ]
    for a in bad:
        assert lib.vox_create(ctypes.byref(c), *a) == -1, a
        assert not c.value
    assert lib.vox_create(ctypes.byref(c), 32, 32, 32, 1 << 21, E, E, 1) == -2  # extent > 2^20
    assert lib.vox_create(None, 32, 32, 32, E, E, E, 1) == -1
    batch = ctypes.c_void_p()
    assert lib.vox_create(ctypes.byref(batch), 64, 64, 64, E, E, E, 256) == 0
    assert lib.vox_grid_words(batch) == 256 * 64 * 64 * 2
    # batch > 1 needs offsets
    assert lib.vox_tets(batch, ctypes.c_void_p(256), 10, ctypes.c_void_p(256), 10, None) == -1
    lib.vox_destroy(batch)


def test_strerror(lib):
    seen = set()
    for code in range(0, -7, -1):
        s = lib.vox_strerror(code).decode()
        assert s and s != "unknown error"
        seen.add(s)
    assert len(seen) == 7
    assert lib.vox_strerror(-99).decode() == "unknown error"


def test_no_cpu_fallback_without_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np

    import paper_2106_01326_b200 as pkg

    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pkg.voxelize(np.zeros((4, 3), np.int32), np.zeros((1, 4), np.int32), (32, 32, 32))


def test_product_does_not_import_oracle():
    pkg_dir = os.path.join(ROOT, "paper_2106_01326_b200")
    for dirpath, _d, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                s = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in s.replace("no CPU oracle", ""), f
