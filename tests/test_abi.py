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


def test_misaligned_workspace_variant_and_tile_count_limits(lib):
    c = ctypes.c_void_p()
    E = 65536
    assert lib.vox_create(ctypes.byref(c), 64, 64, 64, E, E, E, 1) == 0
    assert lib.vox_tets(c, ctypes.c_void_p(256), 4, ctypes.c_void_p(256), 0, None) == 0
    # a workspace that is not 16-byte aligned is refused before anything is enqueued (uint2 / uint4 accesses)
    assert lib.vox_run(c, None, ctypes.c_void_p(256 + 4), 1 << 20, ctypes.c_void_p(256)) == -1
    assert lib.vox_plan(c, None, ctypes.c_void_p(256 + 8), 1 << 20, None) == -1
    assert lib.vox_validate(c, None, ctypes.c_void_p(256 + 4), 1 << 20) == -1
    # variants: 0 default, 1 binned lattice path, 2 fused lattice path; anything else is refused, not ignored
    assert lib.vox_set_variant(c, 0) == 0
    assert lib.vox_set_variant(c, 1) == 0
    assert lib.vox_set_variant(c, 2) == 0
    assert lib.vox_set_variant(c, 3) == -1
    assert lib.vox_set_variant(c, -1) == -1
    assert lib.vox_path(c) == 0  # explicit tets: the binning passes
    # lattice input: the default bins ordinary cells and fuses giant ones; 1 and 2 force either
    assert lib.vox_set_variant(c, 0) == 0
    assert lib.vox_lattice(c, ctypes.c_void_p(256), 8, 8, 8, ctypes.c_void_p(256)) == 0
    assert lib.vox_path(c) == 1           # 64^3 voxels / 8^3 cells: cells of 8 voxels
    assert lib.vox_set_variant(c, 2) == 0 and lib.vox_path(c) == 2
    assert lib.vox_set_variant(c, 1) == 0 and lib.vox_path(c) == 1
    assert lib.vox_set_variant(c, 0) == 0
    assert lib.vox_lattice(c, ctypes.c_void_p(256), 1, 1, 1, ctypes.c_void_p(256)) == 0
    assert lib.vox_path(c) == 2           # one cell of 64^3 voxels: giant
    lib.vox_destroy(c)
    # one CTA per tile: more than 2^31 - 1 tiles cannot be launched -> VOX_ERANGE at create / set_tile
    assert lib.vox_create(ctypes.byref(c), 32768, 4096, 4096, E, E, E, 1000) == -2
    assert not c.value
    assert lib.vox_create(ctypes.byref(c), 32768, 4096, 4096, E, E, E, 100) == 0
    assert lib.vox_set_tile(c, 4, 4) == -2
    assert lib.vox_set_tile(c, 32, 32) == 0
    lib.vox_destroy(c)
    assert lib.vox_kernel_launches() == 0   # callable without a device; nothing was launched by the calls above


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


def _tile(lib, grid, batch, T):
    c = ctypes.c_void_p()
    E = 65536
    assert lib.vox_create(ctypes.byref(c), *grid, E, E, E, batch) == 0
    fake = ctypes.c_void_p(256)  # never dereferenced by vox_tets
    off = fake if batch > 1 else None
    assert lib.vox_tets(c, fake, 10, fake, T, off) == 0
    o = (ctypes.c_int * 5)()
    assert lib.vox_tile_shape(c, o) == 0
    fixed = lib.vox_workspace_fixed_bytes(c)
    lib.vox_destroy(c)
    return tuple(o), fixed


def test_tile_choice_depends_on_grid_and_tet_count(lib):
    """auto_tile: 32^3 bricks for big grids, thinner tiles while there are fewer than
    four waves of CTAs or more than ~1024 tets per tile; a tile fixed by vox_set_tile is kept."""
    (ty, tz, nbx, nby, nbz), _ = _tile(lib, (1024, 1024, 1024), 1, 4829739)     # cfg4
    assert (ty, tz) == (32, 32) and (nbx, nby, nbz) == (32, 32, 32)
    (ty, tz, *_), _ = _tile(lib, (256, 256, 256), 1, 10110954)                    # 10^7 tets at 256^3: min tile
    assert (ty, tz) == (8, 8)
    (ty, tz, nbx, nby, nbz), _ = _tile(lib, (64, 64, 64), 256, 5271425)           # cfg3
    assert 256 * nbx * nby * nbz >= 4 * 1184 and max(ty, tz) <= 16
    (ty, tz, *_), _ = _tile(lib, (32, 32, 32), 1, 384)                            # cfg1: as many CTAs as possible
    assert (ty, tz) == (8, 8)
    small, f_small = _tile(lib, (512, 512, 512), 1, 1000)
    big, f_big = _tile(lib, (512, 512, 512), 1, 40_000_000)
    assert small[0] * small[1] >= big[0] * big[1] and f_big > f_small           # more tets -> thinner tiles
    # a user-fixed tile survives vox_tets
    c = ctypes.c_void_p()
    assert lib.vox_create(ctypes.byref(c), 256, 256, 256, 65536, 65536, 65536, 1) == 0
    assert lib.vox_set_tile(c, 32, 16) == 0
    assert lib.vox_tets(c, ctypes.c_void_p(256), 10, ctypes.c_void_p(256), 10_000_000, None) == 0
    o = (ctypes.c_int * 5)()
    assert lib.vox_tile_shape(c, o) == 0 and (o[0], o[1]) == (32, 16)
    lib.vox_destroy(c)


def test_sparse_and_pipe_argument_checks(lib):
    c = ctypes.c_void_p()
    assert lib.vox_create(ctypes.byref(c), 64, 64, 64, 65536, 65536, 65536, 1) == 0
    fake = ctypes.c_void_p(256)
    assert lib.vox_run_sparse(c, None, fake, 1 << 20, None, fake, 4) == -1          # no table
    assert lib.vox_run_sparse(c, None, fake, 1 << 20, fake, None, 4) == -1          # capacity without payload
    assert lib.vox_run_sparse(c, None, fake, 1 << 20, fake, fake, 4) == -5          # before vox_tets
    assert lib.vox_tile_shape(c, None) == -1
    lib.vox_destroy(c)
    p = ctypes.c_void_p()
    assert lib.vox_pipe_create(ctypes.byref(p), 64, 64, 64, 65536, 65536, 65536, 1, 0, 10, 10) == -1   # depth
    assert lib.vox_pipe_create(ctypes.byref(p), 64, 64, 64, 65536, 65536, 65536, 1, 9, 10, 10) == -1
    assert lib.vox_pipe_create(ctypes.byref(p), 60, 64, 64, 65536, 65536, 65536, 1, 2, 10, 10) == -1   # nx % 32
    assert not p.value
    assert lib.vox_pipe_arena_bytes(None) == 0 and lib.vox_pipe_wait(None, 0, None) == -1
