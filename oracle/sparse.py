"""Oracle for the sparse (two-level) output.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The encoding is defined in include/vox.h ("Sparse (two-level) output"; the paper only says that
"voxels are often calculated and stored in octree data formats"): the dense
grid is cut into tiles of 32 x TY x TZ voxels; a tile whose voxels inside the grid are all empty
gets table word 0, all solid 0xFFFFFFFF, anything else is MIXED and carries its TZ x TY row words
as a payload.  Which payload slot a mixed tile gets is NOT unique (any permutation is valid), so
this module works with what is unique: the per-tile class, the payload CONTENT keyed by tile, and
the decoded dense grid.

Plain loops over tiles on the dense uint32 grid [batch][nz][ny][nx/32] (one word = one x-run of
32 voxels = the x-extent of a tile); nothing here is shared with the CUDA path.
"""
from __future__ import annotations

import numpy as np

EMPTY = 0
FULL = 0xFFFFFFFF
DROPPED = 0xFFFFFFFE
MIXED = 1  # class label used by classify(); a table stores 1 + slot instead


def tiles_per_axis(grid, ty, tz):
    nx, ny, nz = grid
    return nx // 32, -(-ny // ty), -(-nz // tz)


def classify(dense: np.ndarray, ty: int, tz: int):
    """dense uint32[batch][nz][ny][nx/32] -> (cls uint32[NB] in {EMPTY, FULL, MIXED},
    payloads {tile index: uint32[tz][ty]}) following the definition word by word."""
    batch, nz, ny, wpr = dense.shape
    nbx, nby, nbz = wpr, -(-ny // ty), -(-nz // tz)
    cls = np.zeros(batch * nbz * nby * nbx, dtype=np.uint32)
    payloads = {}
    for m in range(batch):
        for bz in range(nbz):
            for by in range(nby):
                z0, y0 = bz * tz, by * ty
                block = dense[m, z0:z0 + tz, y0:y0 + ty, :]  # rows inside the grid only
                for bx in range(nbx):
                    t = ((m * nbz + bz) * nby + by) * nbx + bx
                    w = block[:, :, bx]
                    if not w.any():
                        cls[t] = EMPTY
                    elif np.all(w == np.uint32(FULL)):
                        cls[t] = FULL
                    else:
                        cls[t] = MIXED
                        p = np.zeros((tz, ty), dtype=np.uint32)  # rows outside the grid are 0
                        p[: w.shape[0], : w.shape[1]] = w
                        payloads[t] = p
    return cls, payloads


def decode(table: np.ndarray, payload: np.ndarray, grid, batch: int, ty: int, tz: int) -> np.ndarray:
    """table uint32[NB], payload uint32[>=mixed][tz][ty] -> dense uint32[batch][nz][ny][nx/32]."""
    nx, ny, nz = grid
    nbx, nby, nbz = tiles_per_axis(grid, ty, tz)
    table = np.asarray(table).view(np.uint32).reshape(-1)
    payload = np.asarray(payload).view(np.uint32).reshape(-1, tz, ty)
    assert table.size == batch * nbz * nby * nbx
    dense = np.zeros((batch, nz, ny, nx // 32), dtype=np.uint32)
    for m in range(batch):
        for bz in range(nbz):
            for by in range(nby):
                z0, y0 = bz * tz, by * ty
                hz, hy = min(tz, nz - z0), min(ty, ny - y0)
                for bx in range(nbx):
                    code = int(table[((m * nbz + bz) * nby + by) * nbx + bx])
                    if code == EMPTY:
                        continue
                    if code == FULL:
                        dense[m, z0:z0 + hz, y0:y0 + hy, bx] = np.uint32(FULL)
                    elif code == DROPPED:
                        raise ValueError("table holds a dropped tile")
                    else:
                        dense[m, z0:z0 + hz, y0:y0 + hy, bx] = payload[code - 1, :hz, :hy]
    return dense


def check_table(table: np.ndarray, payload: np.ndarray, dense_expected: np.ndarray, ty: int, tz: int):
    """Everything that is unique about a (table, payload) pair, against the expected dense grid:
    per-tile class, slots = a permutation of 0..mixed-1, payload content per tile (incl. the zero
    rows outside the grid).  Returns the number of mixed tiles; raises AssertionError otherwise."""
    table = np.asarray(table).view(np.uint32).reshape(-1)
    cls, payloads = classify(dense_expected, ty, tz)
    assert table.size == cls.size, (table.size, cls.size)
    got_cls = np.where((table == EMPTY) | (table == np.uint32(FULL)), table, np.uint32(MIXED))
    bad = np.flatnonzero(got_cls != cls)
    assert bad.size == 0, f"{bad.size} tiles misclassified, first tile {bad[:1]}: got {table[bad[:1]]}, want class {cls[bad[:1]]}"
    mixed = np.flatnonzero(cls == MIXED)
    slots = table[mixed].astype(np.int64) - 1
    assert sorted(slots.tolist()) == list(range(mixed.size)), "payload slots are not a permutation of 0..mixed-1"
    payload = np.asarray(payload).view(np.uint32).reshape(-1, tz, ty)
    for t, s in zip(mixed.tolist(), slots.tolist()):
        if not np.array_equal(payload[s], payloads[t]):
            raise AssertionError(f"payload of tile {t} (slot {s}) differs")
    return int(mixed.size)
