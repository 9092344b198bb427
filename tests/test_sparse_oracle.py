"""Pins of oracle/sparse.py (the two-level encoding of include/vox.h) against things fixed
independently of it: hand-built tables, closed-form tile counts of axis-aligned boxes, the
all-ones invariant on ragged grids, and round trips through hand-permuted slots.  CPU only."""
import numpy as np
import pytest

import meshgen
import oracle
from oracle import sparse

F = np.uint32(0xFFFFFFFF)


def test_hand_built_grid_classes_and_payload():
    # grid 64 x 8 x 8, tiles 32 x 4 x 4 -> nbx=2, nby=2, nbz=2: 8 tiles, t = (bz*2 + by)*2 + bx
    d = np.zeros((1, 8, 8, 2), dtype=np.uint32)
    d[0, 0:4, 0:4, 0] = F            # tile 0 (bz0,by0,bx0): full
    d[0, 5, 6, 1] = 0x00010000       # tile 7 (bz1,by1,bx1): one voxel x=32+16, y=6, z=5
    d[0, 0:4, 4:8, 1] = F            # tile 3 (bz0,by1,bx1): full ...
    d[0, 2, 5, 1] = 0x7FFFFFFF       # ... except one voxel -> mixed
    cls, pay = sparse.classify(d, 4, 4)
    assert cls.tolist() == [sparse.FULL, 0, 0, sparse.MIXED, 0, 0, 0, sparse.MIXED]
    assert sorted(pay) == [3, 7]
    want7 = np.zeros((4, 4), np.uint32)
    want7[1, 2] = 0x00010000         # local z = 5-4, local y = 6-4
    assert np.array_equal(pay[7], want7)
    want3 = np.full((4, 4), F)
    want3[2, 1] = 0x7FFFFFFF
    assert np.array_equal(pay[3], want3)
    # a table written by hand with the slots in the "wrong" order still decodes to d
    table = np.array([0xFFFFFFFF, 0, 0, 2, 0, 0, 0, 1], dtype=np.uint32)
    payload = np.stack([want7, want3])
    assert np.array_equal(sparse.decode(table, payload, (64, 8, 8), 1, 4, 4), d)
    assert sparse.check_table(table, payload, d, 4, 4) == 2
    with pytest.raises(AssertionError):      # same slot twice
        sparse.check_table(np.array([0xFFFFFFFF, 0, 0, 1, 0, 0, 0, 1], np.uint32), payload, d, 4, 4)
    with pytest.raises(AssertionError):      # swapped payloads
        sparse.check_table(table, payload[::-1], d, 4, 4)
    with pytest.raises(AssertionError):      # a full tile reported empty
        sparse.check_table(np.array([0, 0, 0, 2, 0, 0, 0, 1], np.uint32), payload, d, 4, 4)


@pytest.mark.parametrize("ty,tz", [(32, 32), (8, 8), (16, 4)])
def test_axis_aligned_box_closed_form(ty, tz):
    """Oracle grid of a Kuhn-subdivided box (pin P3: the set bits are an index box).  Per axis the
    tiles meeting [i0,i1] number floor(i1/s) - floor(i0/s) + 1 and those contained in it can be
    counted the same way; FULL = product of contained, MIXED = product of meeting - FULL."""
    E, n = 65536, 64
    h = E // n
    lo, hi = (5 * h, 16 * h, 0), (40 * h, 48 * h, 31 * h + h // 2)
    cs = [np.array([lo[a], (lo[a] + hi[a]) // 2, hi[a]]) for a in range(3)]
    v, t = meshgen.kuhn.kuhn_mesh(cs[0], cs[1], cs[2], 0.0, None)
    dense = oracle.voxelize(v, t, (n, n, n), (E, E, E))
    size = (32, ty, tz)
    meet, inside = [], []
    for a in range(3):
        i0 = -((h // 2 - lo[a]) // h)            # ceil((lo - h/2)/h)
        i1 = (hi[a] - h // 2) // h
        s = size[a]
        meet.append(i1 // s - i0 // s + 1)
        inside.append(sum(1 for b in range(n // s) if i0 <= b * s and b * s + s - 1 <= i1))
    cls, pay = sparse.classify(dense, ty, tz)
    full = int(np.sum(cls == np.uint32(sparse.FULL)))
    mixed = int(np.sum(cls == sparse.MIXED))
    assert full == inside[0] * inside[1] * inside[2]
    assert mixed == meet[0] * meet[1] * meet[2] - full == len(pay)
    assert int(np.sum(cls == 0)) == cls.size - full - mixed


def test_all_ones_on_a_ragged_grid_is_all_full():
    # ny = 20 and nz = 12 are not multiples of the tile: rows outside the grid must not count
    d = np.full((2, 12, 20, 3), F, dtype=np.uint32)
    cls, pay = sparse.classify(d, 8, 8)
    assert cls.size == 2 * 2 * 3 * 3 and np.all(cls == F) and not pay
    d[1, 11, 19, 2] = 0x7FFFFFFF
    cls, pay = sparse.classify(d, 8, 8)
    t = ((1 * 2 + 1) * 3 + 2) * 3 + 2
    assert list(pay) == [t] and cls[t] == sparse.MIXED
    assert pay[t][3, 3] == 0x7FFFFFFF and np.all(pay[t][4:, :] == 0) and np.all(pay[t][:, 4:] == 0)


def test_cfg1_conforming_box_is_all_full_tiles():
    m = meshgen.make_config("cfg1")  # pin P4: every bit set
    dense = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
    for ty, tz in [(32, 32), (8, 8)]:
        cls, pay = sparse.classify(dense, ty, tz)
        assert np.all(cls == F) and not pay


@pytest.mark.parametrize("shape,ty,tz", [((1, 16, 16, 2), 8, 8), ((3, 10, 7, 1), 4, 4), ((2, 33, 40, 2), 32, 16)])
def test_round_trip_with_permuted_slots(shape, ty, tz):
    rng = np.random.default_rng(sum(shape) + ty)
    d = rng.integers(0, 2**32, shape, dtype=np.uint64).astype(np.uint32)
    d[rng.random(shape) < 0.4] = 0
    d[rng.random(shape) < 0.3] = F
    b, nz, ny, wpr = shape
    cls, pay = sparse.classify(d, ty, tz)
    tiles = sorted(pay)
    perm = rng.permutation(len(tiles))
    table = cls.copy()
    payload = np.zeros((len(tiles) + 2, tz, ty), np.uint32)
    for t, s in zip(tiles, perm.tolist()):
        table[t] = s + 1
        payload[s] = pay[t]
    assert np.array_equal(sparse.decode(table, payload, (wpr * 32, ny, nz), b, ty, tz), d)
    assert sparse.check_table(table, payload, d, ty, tz) == len(tiles)
    # popcount is preserved tile by tile: FULL tiles count their in-grid voxels only
    bits = int(np.unpackbits(d.view(np.uint8)).sum())
    full_bits = 0
    nbx, nby, nbz = sparse.tiles_per_axis((wpr * 32, ny, nz), ty, tz)
    for t in np.flatnonzero(cls == F).tolist():
        by, bz = (t // nbx) % nby, (t // (nbx * nby)) % nbz
        full_bits += 32 * min(ty, ny - by * ty) * min(tz, nz - bz * tz)
    pay_bits = sum(int(np.unpackbits(p.view(np.uint8)).sum()) for p in pay.values())
    assert bits == full_bits + pay_bits
