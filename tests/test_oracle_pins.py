"""Pins for the CPU oracle (``oracle/``): everything here is fixed by the paper
or by mathematics, never by the oracle itself or by the CUDA path.

P1  hand-counted single tet              tests/golden/p1_single_tet.txt
P2  closed form C(m+2,3) for a Kuhn simplex of m voxels per edge
P3  closed form for a Kuhn-subdivided axis-aligned box (index box, product count)
P4  conforming mesh of the closed box [0,E]^3 sets every bit (cfg1, jittered)
P5  predicate identities: Da-Db+Dc-Dd = 6V for every P; vertex / centroid cases
P6  symmetries: vertex permutation, tet order, mirror, axis swap, translation
P7  monotonicity and idempotence of OR
P8  float64 barycentric solve (numpy.linalg.solve) away from the boundary
P9  pure-Python big-integer brute force without bounding boxes; C mode 1
P10 volume sanity
Citations: Theorem 1; Lemma 1.1; Lemma 1.2
PAPER.md:181-185; bounding-box iteration PAPER.md:98.
"""
import itertools
import math
import os

import numpy as np
import pytest

import meshgen
import oracle
from meshgen.kuhn import kuhn_mesh

E = 65536
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def unpack(bits):
    """uint32[..][nz][ny][nx/32] -> bool[..][nz][ny][nx] (LSB = lowest x)."""
    b = np.ascontiguousarray(bits).view(np.uint8)
    return np.unpackbits(b, axis=-1, bitorder="little").astype(bool)


def popcount(bits):
    return int(unpack(bits).sum())


KUHN_TET = [(0, 0, 0), (1, 0, 0), (1, 1, 0), (1, 1, 1)]  # {0 <= z <= y <= x <= 1}


# ----------------------------------------------------------------------------- P1
def test_p1_hand_counted_single_tet():
    expect = np.zeros((32, 32, 1), dtype=np.uint32)
    with open(os.path.join(GOLDEN, "p1_single_tet.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            z, y, w = line.split()
            expect[int(z), int(y), 0] = int(w, 16)
    m = meshgen.single_tet_mesh(*[tuple(8192 * c for c in v) for v in KUHN_TET])
    got = oracle.voxelize(m.verts, m.tets, m.grid)[0]
    assert popcount(expect) == 20
    assert np.array_equal(got, expect)
    # every one of the 24 vertex orders (both orientation types, Lemma 1.1) gives the same grid
    for perm in itertools.permutations(range(4)):
        got = oracle.voxelize(m.verts, m.tets[:, list(perm)], m.grid)[0]
        assert np.array_equal(got, expect), perm


# ----------------------------------------------------------------------------- P2
@pytest.mark.parametrize("m_vox", [1, 2, 3, 4, 8, 32])
def test_p2_kuhn_simplex_closed_form(m_vox):
    h = 2048
    L = m_vox * h
    for axes in itertools.permutations(range(3)):
        vs = []
        for v in KUHN_TET:
            p = [0, 0, 0]
            for src, dst in enumerate(axes):
                p[dst] = v[src] * L
            vs.append(tuple(p))
        m = meshgen.single_tet_mesh(*vs)
        got = oracle.voxelize(m.verts, m.tets, m.grid)
        assert popcount(got) == math.comb(m_vox + 2, 3), (m_vox, axes)
    assert math.comb(32 + 2, 3) == 5984


def test_p2_strict_reading_would_differ():
    # Reading G1: Theorem 1's strict test leaves holes on shared faces.  One Kuhn cell
    # [0,4h]^3: inclusive 64/64, strict 24/64 (points with three distinct coordinates).
    h = 2048
    v, t = kuhn_mesh([0, 4 * h], [0, 4 * h], [0, 4 * h], 0.0, None)
    grid, ext = (32, 4, 4), (E, 4 * h, 4 * h)
    inc = oracle.bruteforce_voxelize(v, t, grid, ext)
    strict = oracle.bruteforce_voxelize(v, t, grid, ext, strict=True)
    assert popcount(inc) == 64 and popcount(strict) == 24
    assert np.array_equal(oracle.voxelize(v, t, grid, ext)[0], inc)


# ----------------------------------------------------------------------------- P3
@pytest.mark.parametrize(
    "lo,hi,cells",
    [((0, 0, 0), (E, E, E), (1, 1, 1)),
     ((3000, 5000, 7000), (40000, 33000, 60001), (3, 2, 4)),
     ((1024, 1024, 1024), (1024 + 2048 * 5, 1024 + 2048 * 7, 3072), (2, 3, 1)),
     ((1025, 1023, 10), (9000, 9216, 1023), (1, 2, 1))],
)
def test_p3_kuhn_box_closed_form(lo, hi, cells):
    h, n = 2048, 32
    cs = [np.rint(np.linspace(lo[k], hi[k], cells[k] + 1)).astype(np.int64) for k in range(3)]
    v, t = kuhn_mesh(cs[0], cs[1], cs[2], 0.0, None)
    got = unpack(oracle.voxelize(v, t, (n, n, n))[0])  # [z][y][x]
    expect = np.zeros((n, n, n), dtype=bool)
    rng = []
    for k in range(3):
        i0 = max(0, -((-(2 * lo[k] - h)) // (2 * h)))  # ceil((lo-h/2)/h)
        i1 = min(n - 1, (2 * hi[k] - h) // (2 * h))  # floor((hi-h/2)/h)
        rng.append((i0, i1))
    (x0, x1), (y0, y1), (z0, z1) = rng
    if x0 <= x1 and y0 <= y1 and z0 <= z1:
        expect[z0 : z1 + 1, y0 : y1 + 1, x0 : x1 + 1] = True
    assert np.array_equal(got, expect)
    assert got.sum() == max(0, x1 - x0 + 1) * max(0, y1 - y0 + 1) * max(0, z1 - z0 + 1)


def test_p3_union_not_sum():
    # one cube of m voxels per edge: union m^3, while the six tets sum to 6*C(m+2,3)
    h, m_vox = 2048, 4
    v, t = kuhn_mesh([0, m_vox * h], [0, m_vox * h], [0, m_vox * h], 0.0, None)
    whole = popcount(oracle.voxelize(v, t, (32, 32, 32)))
    parts = sum(popcount(oracle.voxelize(v, t[i : i + 1], (32, 32, 32))) for i in range(6))
    assert whole == m_vox ** 3
    assert parts == 6 * math.comb(m_vox + 2, 3)


# ----------------------------------------------------------------------------- P4
@pytest.mark.parametrize("name", ["cfg1", "s1"])
def test_p4_conforming_box_all_ones(name):
    m = meshgen.make_config(name)
    assert m.expect_all_ones
    got = oracle.voxelize(m.verts, m.tets, m.grid)
    assert np.all(got == np.uint32(0xFFFFFFFF))


def test_p4_other_grids_and_cells():
    rng = np.random.default_rng(7)
    c = np.rint(np.arange(25) * E / 24).astype(np.int64)  # 24 cells: non-integer cell width
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    got = oracle.voxelize(v, t, (64, 64, 64))
    assert np.all(got == np.uint32(0xFFFFFFFF))
    # anisotropic grid and extent
    v, t = kuhn_mesh(np.arange(0, 4097, 512), np.arange(0, 8193, 1024), [0, 100, 300, 1024], 0.2, rng)
    got = oracle.voxelize(v, t, (64, 16, 8), extent=(4096, 8192, 1024))
    assert np.all(got == np.uint32(0xFFFFFFFF))


# ----------------------------------------------------------------------------- P5
def test_p5_predicate_identities():
    rng = np.random.default_rng(11)
    for _ in range(500):
        A, B, C, D, P = (rng.integers(0, E + 1, 3) for _ in range(5))
        Da, Db, Dc, Dd, V6 = oracle.determinants(P, A, B, C, D)
        # Lemma 1.2: the four D are the signed volumes of PBCD, PACD, PABD, PABC
        assert Da - Db + Dc - Dd == V6
        # independent 6V with Python integers
        u, v, w = (B - A).tolist(), (C - A).tolist(), (D - A).tolist()
        V6_py = (u[0] * (v[1] * w[2] - v[2] * w[1]) - u[1] * (v[0] * w[2] - v[2] * w[0])
                 + u[2] * (v[0] * w[1] - v[1] * w[0]))
        assert V6 == V6_py
        if V6 == 0:
            continue
        # P = a vertex: three of the four vanish and the inclusive test is true
        for k, Q in enumerate((A, B, C, D)):
            d = oracle.determinants(Q, A, B, C, D)[:4]
            assert sum(1 for x in d if x == 0) >= 3 and abs(d[k]) == abs(V6)
            assert oracle.inside(Q, A, B, C, D)


def test_p5_centroid_without_fractions():
    rng = np.random.default_rng(12)
    n = 0
    while n < 200:
        A0, B0, C0, D0 = (rng.integers(0, 16384, 3) for _ in range(4))
        A, B, C, D = 4 * A0, 4 * B0, 4 * C0, 4 * D0
        P = A0 + B0 + C0 + D0  # centroid of the scaled tet, an integer point
        Da, Db, Dc, Dd, V6 = oracle.determinants(P, A, B, C, D)
        if V6 == 0:
            continue
        n += 1
        assert abs(Da) == abs(Db) == abs(Dc) == abs(Dd) == abs(V6) // 4 and abs(V6) % 4 == 0
        assert (Da > 0) == (Dc > 0) == (V6 > 0) and (Db > 0) == (Dd > 0) == (V6 < 0)
        assert oracle.inside(P, A, B, C, D)
        # reflecting the centroid through a vertex puts it strictly outside
        assert not oracle.inside(np.clip(2 * A - P, -2**30, 2**30), A, B, C, D)


def test_p5_degenerate_tets_contribute_nothing():
    # reading G2: four coplanar points, or a repeated vertex
    v = np.array([[0, 0, 1024], [E, 0, 1024], [0, E, 1024], [E, E, 1024]], dtype=np.int32)
    t = np.array([[0, 1, 2, 3], [0, 1, 2, 2], [1, 1, 1, 1]], dtype=np.int32)
    got = oracle.voxelize(v, t, (32, 32, 32))
    assert popcount(got) == 0
    assert popcount(oracle.voxelize(v, t, (32, 32, 32), mode=1)) == 0


# ----------------------------------------------------------------------------- P6
def _small_carved(seed=21, cells=5, lo=8192, hi=8192 + 5 * 6144):
    rng = np.random.default_rng(seed)
    c = np.rint(np.linspace(lo, hi, cells + 1)).astype(np.int64)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    keep = rng.random(len(t)) < 0.6
    return v, t[keep]


def test_p6_symmetries():
    rng = np.random.default_rng(22)
    v, t = _small_carved()
    grid = (32, 32, 32)
    base = oracle.voxelize(v, t, grid)[0]
    vox = unpack(base)
    assert 0 < vox.sum() < vox.size
    # vertex order within each tet (both orientation types)
    tp = t.copy()
    for i in range(len(tp)):
        tp[i] = tp[i][rng.permutation(4)]
    assert np.array_equal(oracle.voxelize(v, tp, grid)[0], base)
    # tet order
    assert np.array_equal(oracle.voxelize(v, t[rng.permutation(len(t))], grid)[0], base)
    # mirror c -> E - c per axis
    for axis in range(3):
        vm = v.copy()
        vm[:, axis] = E - vm[:, axis]
        got = unpack(oracle.voxelize(vm, t, grid)[0])
        assert np.array_equal(got, np.flip(vox, axis=2 - axis)), axis
    # swapping two coordinate axes transposes the grid
    for a, b in [(0, 1), (0, 2), (1, 2)]:
        vs = v.copy()
        vs[:, [a, b]] = vs[:, [b, a]]
        got = unpack(oracle.voxelize(vs, t, grid)[0])
        assert np.array_equal(got, np.swapaxes(vox, 2 - a, 2 - b)), (a, b)
    # translation by a multiple of the pitch shifts the grid
    h = 2048
    for shift in [(3, 0, 0), (0, -2, 0), (1, 2, -3)]:
        vt = v + np.array(shift, dtype=np.int32) * h
        got = unpack(oracle.voxelize(vt, t, grid)[0])
        exp = np.roll(vox, shift=(shift[2], shift[1], shift[0]), axis=(0, 1, 2))
        assert np.array_equal(got, exp), shift


# ----------------------------------------------------------------------------- P7
def test_p7_monotone_and_idempotent():
    v, t = _small_carved(seed=31)
    grid = (32, 32, 32)
    full = unpack(oracle.voxelize(v, t, grid)[0])
    part = unpack(oracle.voxelize(v, t[::2], grid)[0])
    assert np.all(full[part])  # removing tets only clears bits
    dup = unpack(oracle.voxelize(v, np.concatenate([t, t, t[::3]]), grid)[0])
    assert np.array_equal(dup, full)


# ----------------------------------------------------------------------------- P8
def test_p8_float_barycentric_away_from_boundary():
    rng = np.random.default_rng(41)
    checked = 0
    n_in = 0
    for _ in range(400):
        A, B, C, D = (rng.integers(0, E + 1, 3) for _ in range(4))
        M = np.stack([A - D, B - D, C - D], axis=1).astype(np.float64)
        if abs(np.linalg.det(M)) < 1e3:
            continue
        lo, hi = np.minimum.reduce([A, B, C, D]), np.maximum.reduce([A, B, C, D])
        for _p in range(20):
            P = rng.integers(lo, hi + 1)
            lam3 = np.linalg.solve(M, (P - D).astype(np.float64))
            lam = np.append(lam3, 1.0 - lam3.sum())
            if np.min(np.abs(lam)) < 1e-9:
                continue
            checked += 1
            expect = bool(np.all(lam > 0))
            n_in += expect
            assert oracle.inside(P, A, B, C, D) == expect
    assert checked > 5000 and n_in > 300


# ----------------------------------------------------------------------------- P9
def test_p9_bruteforce_python_cfg1_shaped():
    # config-1 mesh on a thinner grid so that pure Python finishes in seconds
    m = meshgen.make_config("cfg1")
    grid = (32, 8, 4)
    bf = oracle.bruteforce_voxelize(m.verts, m.tets, grid)
    assert np.all(bf == np.uint32(0xFFFFFFFF))
    assert np.array_equal(oracle.voxelize(m.verts, m.tets, grid)[0], bf)


@pytest.mark.parametrize("seed", [51, 52, 53])
def test_p9_bruteforce_python_random_carved(seed):
    rng = np.random.default_rng(seed)
    c = np.array([0, 30000 + seed, E])
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    # jitter the boundary too, so tets stick out less regularly; keep inside [0,E]
    v = np.clip(v + rng.integers(-3000, 3001, v.shape), 0, E).astype(np.int32)
    t = t[rng.random(len(t)) < 0.7]
    grid = (32, 16, 8)
    bf = oracle.bruteforce_voxelize(v, t, grid)
    assert 0 < popcount(bf) < 32 * 16 * 8
    assert np.array_equal(oracle.voxelize(v, t, grid, mode=0)[0], bf)
    assert np.array_equal(oracle.voxelize(v, t, grid, mode=1)[0], bf)


def test_p9_mode1_equals_mode0_bbox_rounding():
    # vertices exactly on voxel centres and on voxel faces stress the closed-bbox rounding (G8)
    rng = np.random.default_rng(61)
    h = 2048
    pts = (rng.integers(0, 65, (40, 3)) * (h // 2)).astype(np.int32)  # multiples of h/2 in [0,E]
    t = np.array([rng.choice(40, 4, replace=False) for _ in range(60)], dtype=np.int32)
    a = oracle.voxelize(pts, t, (32, 32, 32), mode=0)
    b = oracle.voxelize(pts, t, (32, 32, 32), mode=1)
    assert np.array_equal(a, b) and popcount(a) > 0


def test_batch_layout_and_offsets():
    m = meshgen.make_config("cfg3_small")
    got = oracle.voxelize(m.verts, m.tets, m.grid, tet_offsets=m.tet_offsets)
    assert got.shape == (4, 64, 64, 2)
    for k in range(m.batch):
        s, e = m.tet_offsets[k], m.tet_offsets[k + 1]
        one = oracle.voxelize(m.verts, m.tets[s:e], m.grid)[0]
        assert np.array_equal(got[k], one)
    assert len({got[k].tobytes() for k in range(4)}) == 4


# ----------------------------------------------------------------------------- P10
def test_p10_volume_sanity_cfg2():
    m = meshgen.make_config("cfg2")
    got, samples = oracle.voxelize(m.verts, m.tets, m.grid, return_samples=True)
    P = m.verts[m.tets].astype(np.int64)
    u, v, w = P[:, 1] - P[:, 0], P[:, 2] - P[:, 0], P[:, 3] - P[:, 0]
    vol6 = np.abs(np.einsum("ij,ij->i", u, np.cross(v, w)))
    h = E // m.grid[0]
    vol_vox = vol6.sum() / 6.0 / h ** 3
    assert abs(popcount(got) - vol_vox) / vol_vox < 0.02
    assert 50 < samples / m.T < 150  # "only a handful sample candidates" per tet
