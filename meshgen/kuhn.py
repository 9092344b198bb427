"""Jittered Kuhn-subdivision tet meshes on an integer lattice, carved by shape.

Recipe (BASELINE.json configs 1-5):
  * an axis-aligned cell grid with corner coordinates xs[0..cx], ys[0..cy],
    zs[0..cz] on the integer lattice [0, E]^3, E = 65536;
  * vertex id = (i*(cy+1) + j)*(cz+1) + k;
  * 6 tets per cell, one per permutation pi of the axes, vertices listed along
    the path  corner -> +e_pi(1) -> +e_pi(2) -> +e_pi(3)  (so 3 of the 6 tets
    have positive and 3 negative signed volume);
  * jitter: every INTERIOR vertex moves, per coordinate, by
    rint(u * jit * min(adjacent cell widths on that axis)), u ~ U(-1, 1);
    vertices on the box boundary do not move at all (the hull stays the box);
  * carving keeps a tet iff its centroid (float64 mean of its 4 vertices)
    satisfies a shape predicate; vertices are NOT compacted afterwards.

No point-in-tet test, bounding box or voxel grid is computed here.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

E_LATTICE = 65536

_PERMS = list(itertools.permutations(range(3)))  # 6 axis orders


@dataclass
class Mesh:
    """One voxelization job: `batch` independent meshes sharing one grid shape."""

    name: str
    verts: np.ndarray  # int32 [V][3]
    tets: np.ndarray  # int32 [T][4], indices global into verts
    grid: tuple  # (nx, ny, nz) voxels per mesh
    extent: tuple = (E_LATTICE, E_LATTICE, E_LATTICE)
    tet_offsets: np.ndarray = field(default=None)  # int64 [batch+1]
    expect_all_ones: bool = False  # union of the tets is the closed box [0,E]^3
    cells: tuple = None  # (cx, cy, cz) when verts/tets come from kuhn_mesh of that lattice (see lattice_form)

    def __post_init__(self):
        if self.tet_offsets is None:
            self.tet_offsets = np.array([0, len(self.tets)], dtype=np.int64)
        self.verts = np.ascontiguousarray(self.verts, dtype=np.int32)
        self.tets = np.ascontiguousarray(self.tets, dtype=np.int32).reshape(-1, 4)
        self.tet_offsets = np.ascontiguousarray(self.tet_offsets, dtype=np.int64)

    @property
    def batch(self) -> int:
        return len(self.tet_offsets) - 1

    @property
    def T(self) -> int:
        return int(self.tets.shape[0])

    @property
    def V(self) -> int:
        return int(self.verts.shape[0])

    @property
    def grid_words(self) -> int:
        nx, ny, nz = self.grid
        return self.batch * nz * ny * (nx // 32)


def _uniform_corners(n_cells: int, extent: int = E_LATTICE) -> np.ndarray:
    return np.rint(np.arange(n_cells + 1, dtype=np.float64) * extent / n_cells).astype(np.int64)


def kuhn_mesh(xs, ys, zs, jitter: float, rng: np.random.Generator | None):
    """Vertices and the 6-per-cell Kuhn tets of the cell grid xs x ys x zs.

    Returns (verts int32[V][3], tets int32[6*cells][4]); tet order is
    cell-major (i, j, k) then permutation.
    """
    xs = np.asarray(xs, dtype=np.int64)
    ys = np.asarray(ys, dtype=np.int64)
    zs = np.asarray(zs, dtype=np.int64)
    cx, cy, cz = len(xs) - 1, len(ys) - 1, len(zs) - 1
    gx, gy, gz = np.meshgrid(xs, ys, zs, indexing="ij")
    pts = np.stack([gx, gy, gz], axis=-1)  # (cx+1, cy+1, cz+1, 3) int64

    if jitter > 0.0:
        u = rng.uniform(-1.0, 1.0, size=(cx + 1, cy + 1, cz + 1, 3))

        def min_adjacent(c):
            w = np.diff(c).astype(np.float64)
            m = np.empty(len(c))
            m[0], m[-1] = w[0], w[-1]
            m[1:-1] = np.minimum(w[:-1], w[1:])
            return m

        wx, wy, wz = min_adjacent(xs), min_adjacent(ys), min_adjacent(zs)
        scale = np.stack(np.meshgrid(wx, wy, wz, indexing="ij"), axis=-1) * jitter
        d = np.rint(u * scale).astype(np.int64)
        interior = np.zeros((cx + 1, cy + 1, cz + 1), dtype=bool)
        interior[1:-1, 1:-1, 1:-1] = True
        pts = pts + d * interior[..., None]

    verts = pts.reshape(-1, 3).astype(np.int32)

    def vid(i, j, k):
        return (i * (cy + 1) + j) * (cz + 1) + k

    ci, cj, ck = np.meshgrid(np.arange(cx), np.arange(cy), np.arange(cz), indexing="ij")
    ci, cj, ck = ci.ravel(), cj.ravel(), ck.ravel()
    tets = np.empty((ci.size, 6, 4), dtype=np.int64)
    for p, perm in enumerate(_PERMS):
        off = np.zeros(3, dtype=np.int64)
        tets[:, p, 0] = vid(ci, cj, ck)
        for step, axis in enumerate(perm):
            off[axis] += 1
            tets[:, p, step + 1] = vid(ci + off[0], cj + off[1], ck + off[2])
    return verts, tets.reshape(-1, 4).astype(np.int32)


def _centroids(verts, tets):
    return verts[tets].astype(np.float64).mean(axis=1)


def _keep(verts, tets, pred):
    c = _centroids(verts, tets)
    return np.ascontiguousarray(tets[pred(c)])


# ---------------------------------------------------------------- shape predicates
def _in_sphere(c, centre, r):
    return ((c - np.asarray(centre)) ** 2).sum(axis=1) <= r * r


def _in_torus(c, centre, R, r, axis):
    d = c - np.asarray(centre)
    a = d[:, axis]
    o = np.delete(d, axis, axis=1)
    q = np.sqrt((o ** 2).sum(axis=1)) - R
    return q * q + a * a <= r * r


def _in_ellipsoid(c, centre, semi, rot):
    d = (c - centre) @ rot  # into the ellipsoid's frame
    return ((d / semi) ** 2).sum(axis=1) <= 1.0


# ---------------------------------------------------------------- configs
def _cfg1(seed):
    rng = np.random.default_rng(seed)
    c = _uniform_corners(4)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    return Mesh("cfg1_tiny_kuhn4", v, t, (32, 32, 32), expect_all_ones=True, cells=(4, 4, 4))


def _cfg2(seed):
    rng = np.random.default_rng(seed)
    c = _uniform_corners(32)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    E = E_LATTICE
    t = _keep(v, t, lambda p: _in_sphere(p, (E / 2, E / 2, E / 2), 0.45 * E))
    return Mesh("cfg2_sphere_kuhn32", v, t, (128, 128, 128), cells=(32, 32, 32))


def _cfg3_one(seed):
    """One ModelNet-shaped mesh: union of 1-8 random ellipsoids, 15-40k tets.

    The ellipsoid draw is repeated (same generator, so still a pure function of
    the seed) until the kept-tet count lands in BASELINE.json's 15-40k band.
    """
    rng = np.random.default_rng(seed)
    c = _uniform_corners(24)
    v, t_all = kuhn_mesh(c, c, c, 0.2, rng)
    cen = _centroids(v, t_all)
    E = float(E_LATTICE)
    for _ in range(64):
        k = int(rng.integers(1, 9))
        keep = np.zeros(len(t_all), dtype=bool)
        for _e in range(k):
            semi = rng.uniform(0.1, 0.4, size=3) * E
            centre = rng.uniform(0.3, 0.7, size=3) * E
            q, _r = np.linalg.qr(rng.normal(size=(3, 3)))
            keep |= _in_ellipsoid(cen, centre, semi, q)
        n = int(keep.sum())
        if 15000 <= n <= 40000:
            break
    return v, np.ascontiguousarray(t_all[keep])


def _cfg3(seed, n_meshes=256):
    vs, ts, offs = [], [], [0]
    vbase = 0
    for m in range(n_meshes):
        v, t = _cfg3_one(seed + m)
        vs.append(v)
        ts.append(t.astype(np.int64) + vbase)
        vbase += len(v)
        offs.append(offs[-1] + len(t))
    return Mesh(
        f"cfg3_modelnet_batch{n_meshes}",
        np.concatenate(vs),
        np.concatenate(ts).astype(np.int32),
        (64, 64, 64),
        tet_offsets=np.array(offs, dtype=np.int64),
        cells=(24, 24, 24),
    )


def _cfg4(seed, cells=128, grid=1024):
    rng = np.random.default_rng(seed)
    c = _uniform_corners(cells)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    E = float(E_LATTICE)
    # seeded placement of 3 spheres, 2 tori and one box with 4 z-axis through-holes
    sph = [(rng.uniform(0.25, 0.75, 3) * E, rng.uniform(0.20, 0.28) * E) for _ in range(3)]
    tor = [
        (rng.uniform(0.35, 0.65, 3) * E, rng.uniform(0.26, 0.32) * E, rng.uniform(0.08, 0.11) * E, int(rng.integers(0, 3)))
        for _ in range(2)
    ]
    blo = rng.uniform(0.06, 0.12, 3) * E
    bhi = rng.uniform(0.70, 0.94, 3) * E
    bhi[2] = blo[2] + rng.uniform(0.30, 0.38) * E  # a slab-like box
    holes = [
        (blo[:2] + rng.uniform(0.2, 0.8, 2) * (bhi[:2] - blo[:2]), rng.uniform(0.04, 0.08) * E) for _ in range(4)
    ]

    def pred(p):
        keep = np.zeros(len(p), dtype=bool)
        for ctr, r in sph:
            keep |= _in_sphere(p, ctr, r)
        for ctr, R, r, ax in tor:
            keep |= _in_torus(p, ctr, R, r, ax)
        box = np.all((p >= blo) & (p <= bhi), axis=1)
        for hc, hr in holes:
            box &= ((p[:, :2] - hc) ** 2).sum(axis=1) > hr * hr
        return keep | box

    # carve in slabs to bound the float64 centroid temporaries
    parts = []
    step = 1 << 21
    for s in range(0, len(t), step):
        parts.append(_keep(v, t[s : s + step], pred))
    t = np.concatenate(parts)
    return Mesh(f"cfg4_thingi_kuhn{cells}", v, t, (grid, grid, grid), cells=(cells, cells, cells))


def _cfg5(seed):
    """Size/shape stress.  Reading of BASELINE.json's wording: DESIGN.md R-cfg5."""
    rng = np.random.default_rng(seed)
    E = E_LATTICE
    wx = np.rint(32.0 * 1.15 ** np.arange(41)).astype(np.int64)  # 1/4 voxel .. ~67 voxels
    xs = np.concatenate([[0], np.cumsum(wx)])
    xs[-1] = E  # last cell absorbs the remainder
    ys = _uniform_corners(48)
    period = np.array([1024, 512, 256, 128, 64], dtype=np.int64)  # 8,4,2,1,1/2 voxels
    wz = np.tile(period, 33)
    wz = np.concatenate([wz, [E - wz.sum()]])
    zs = np.concatenate([[0], np.cumsum(wz)])
    assert xs[-1] == E and zs[-1] == E and np.all(np.diff(xs) > 0) and np.all(np.diff(zs) > 0)
    v, t = kuhn_mesh(xs, ys, zs, 0.1, rng)
    return Mesh("cfg5_graded_stress", v, t, (512, 512, 512), expect_all_ones=True,
                cells=(len(xs) - 1, len(ys) - 1, len(zs) - 1))


def _s1(seed, jitter=0.2):
    rng = np.random.default_rng(seed)
    c = _uniform_corners(2)
    v, t = kuhn_mesh(c, c, c, jitter, rng)
    return Mesh("s1_giant_tets", v, t, (512, 512, 512), expect_all_ones=True, cells=(2, 2, 2))


def _s2(seed, cells):
    rng = np.random.default_rng(seed)
    c = _uniform_corners(cells)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    return Mesh(f"s2_table1_kuhn{cells}", v, t, (256, 256, 256), expect_all_ones=True, cells=(cells, cells, cells))


_CONFIGS = {
    "cfg1": (lambda s: _cfg1(s), 1001),
    "cfg2": (lambda s: _cfg2(s), 1002),
    "cfg3": (lambda s: _cfg3(s), 3000),
    "cfg3_small": (lambda s: _cfg3(s, n_meshes=4), 3000),
    "cfg4": (lambda s: _cfg4(s), 1004),
    "cfg4_small": (lambda s: _cfg4(s, cells=32, grid=256), 1004),
    "cfg5": (lambda s: _cfg5(s), 1005),
    "s1": (lambda s: _s1(s), 1101),
    "s2_1e5": (lambda s: _s2(s, 26), 1201),
    "s2_1e6": (lambda s: _s2(s, 55), 1202),
    "s2_1e7": (lambda s: _s2(s, 119), 1203),
}


def config_names():
    return list(_CONFIGS)


def make_config(name: str, seed: int | None = None) -> Mesh:
    """Build one of BASELINE.json's configs (cfg1..cfg5) or a supplementary one."""
    fn, default_seed = _CONFIGS[name]
    return fn(default_seed if seed is None else seed)


# ---------------------------------------------------------------- carved variants
def carve_every_third(m: Mesh) -> Mesh:
    """Drop every tet whose index t satisfies t % 3 == 0 (single-mesh jobs only)."""
    assert m.batch == 1
    keep = np.arange(m.T) % 3 != 0
    return Mesh(m.name + "_drop3", m.verts, m.tets[keep], m.grid, m.extent)


def carve_sphere(m: Mesh, frac: float = 0.4) -> Mesh:
    """Keep only tets whose centroid is within frac*E of the box centre."""
    assert m.batch == 1
    ex, ey, ez = m.extent
    t = _keep(m.verts, m.tets, lambda p: _in_sphere(p, (ex / 2, ey / 2, ez / 2), frac * ex))
    return Mesh(m.name + "_sphere", m.verts, t, m.grid, m.extent)


def lattice_form(m: Mesh, cells) -> np.ndarray:
    """keep mask uint8[cx*cy*cz] of a (carved) kuhn_mesh job with `cells` = (cx, cy, cz): bit q of cell c is set iff
    the cell's q-th tet (q = index into the lexicographic permutations of the axes, as kuhn_mesh lists them) is in
    m.tets.  With m.verts this is the lattice input of include/vox.h ("vox_lattice"); m.tets is the same mesh
    written out.  Pure index bookkeeping."""
    cx, cy, cz = (int(c) for c in cells)
    vm = (cx + 1) * (cy + 1) * (cz + 1)
    assert m.V == m.batch * vm
    if m.batch > 1:  # a batch of meshes on the same lattice dims: one block of keep bytes per mesh
        parts = []
        for b in range(m.batch):
            lo, hi = int(m.tet_offsets[b]), int(m.tet_offsets[b + 1])
            one = Mesh(m.name, m.verts[b * vm:(b + 1) * vm], m.tets[lo:hi] - b * vm, m.grid, m.extent)
            parts.append(lattice_form(one, cells))
        return np.concatenate(parts)
    t = m.tets.astype(np.int64)
    v0 = t[:, 0]
    k = v0 % (cz + 1)
    j = (v0 // (cz + 1)) % (cy + 1)
    i = v0 // ((cz + 1) * (cy + 1))
    sx, sy = (cy + 1) * (cz + 1), cz + 1  # vertex-id strides of a step along x, y (z: 1)

    def axis(d):
        return np.where(d == sx, 0, np.where(d == sy, 1, 2))

    a1, a2 = axis(t[:, 1] - t[:, 0]), axis(t[:, 2] - t[:, 1])
    q = _perm_index(a1, a2)
    keep = np.zeros(cx * cy * cz, dtype=np.uint8)
    np.bitwise_or.at(keep, (i * cy + j) * cz + k, (1 << q).astype(np.uint8))
    return keep


def _perm_index(a1, a2):
    table = np.full((3, 3), -1, dtype=np.int64)
    for q, perm in enumerate(_PERMS):
        table[perm[0], perm[1]] = q
    return table[a1, a2]


def single_tet_mesh(a, b, c, d, grid=(32, 32, 32), extent=(E_LATTICE,) * 3) -> Mesh:
    v = np.array([a, b, c, d], dtype=np.int32)
    t = np.array([[0, 1, 2, 3]], dtype=np.int32)
    return Mesh("single_tet", v, t, grid, extent)
