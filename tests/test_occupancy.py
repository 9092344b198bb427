"""Sub-sample occupancy: pins of oracle/occupancy.py (CPU) and GPU parity of vox_occupancy."""
import numpy as np
import pytest

import meshgen
import oracle
from meshgen.kuhn import kuhn_mesh
from oracle.occupancy import occupancy

E = 65536


def _fine(m, k):
    g = tuple(k * n for n in m.grid)
    return oracle.voxelize(m.verts, m.tets, g, m.extent, tet_offsets=m.tet_offsets), g


def test_hand_built_words():
    # one coarse row of 16 voxels at k = 2: fine rows are single words
    d = np.zeros((1, 2, 2, 1), dtype=np.uint32)
    d[0, 0, 0, 0] = 0b1011          # fine x = 0,1,3 of fine row (y=0,z=0)
    d[0, 1, 1, 0] = 0b0110          # fine x = 1,2 of fine row (y=1,z=1)
    d[0, 0, 1, 0] = 0x80000000      # fine x = 31
    c = occupancy(d, 2)
    assert c.shape == (1, 1, 1, 16)
    assert c[0, 0, 0].tolist() == [3, 2] + [0] * 13 + [1]
    d4 = np.zeros((1, 4, 4, 1), dtype=np.uint32)
    d4[0, :, :, 0] = 0x0000F00F     # fine x 0..3 and 12..15 on all 16 fine rows
    assert occupancy(d4, 4)[0, 0, 0].tolist() == [64, 0, 0, 64, 0, 0, 0, 0]


@pytest.mark.parametrize("k", [2, 4])
def test_conforming_box_counts_k_cubed_everywhere(k):
    m = meshgen.make_config("cfg1")                      # pin P4: every fine sample of the closed box is solid
    fine, _ = _fine(m, k)
    c = occupancy(fine, k)
    assert c.shape == (1, 32, 32, 32) and np.all(c == k ** 3)


@pytest.mark.parametrize("k", [2, 4])
def test_axis_aligned_box_is_separable(k):
    """Kuhn box (pin P3: the fine set bits are an index box), so count(x,y,z) = cx(x)*cy(y)*cz(z) with
    c_a(i) = number of fine indices k*i..k*i+k-1 inside [i0_a, i1_a]."""
    n = 32
    hf = E // (n * k)
    lo, hi = (3 * hf + 7, 10 * hf, 0), (41 * hf + 5, 50 * hf + hf // 2, 17 * hf)
    cs = [np.array([lo[a], (lo[a] + hi[a]) // 2, hi[a]]) for a in range(3)]
    v, t = kuhn_mesh(cs[0], cs[1], cs[2], 0.0, None)
    fine = oracle.voxelize(v, t, (n * k,) * 3, (E,) * 3)
    c = occupancy(fine, k)
    per = []
    for a in range(3):
        i0 = -((hf // 2 - lo[a]) // hf)
        i1 = (hi[a] - hf // 2) // hf
        per.append(np.array([sum(1 for f in range(k * i, k * i + k) if i0 <= f <= i1) for i in range(n)]))
    want = per[2][:, None, None] * per[1][None, :, None] * per[0][None, None, :]
    assert np.array_equal(c[0].astype(np.int64), want)
    assert int(c.sum()) == int(np.unpackbits(fine.view(np.uint8)).sum())      # nothing lost, nothing counted twice


def test_total_equals_fine_popcount_and_bounds():
    m = meshgen.carve_sphere(meshgen.make_config("cfg1"))
    for k in (2, 4):
        fine, _ = _fine(m, k)
        c = occupancy(fine, k)
        assert int(c.astype(np.int64).sum()) == int(np.unpackbits(fine.view(np.uint8)).sum())
        assert c.max() <= k ** 3
    # k = 1 is the identity on bits
    d = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
    assert np.array_equal(occupancy(d, 1).reshape(-1), np.unpackbits(d.view(np.uint8), bitorder="little"))


@pytest.mark.gpu
@pytest.mark.parametrize("name,k", [("cfg1", 2), ("cfg1", 4), ("cfg2", 2), ("cfg2", 4), ("cfg3_small", 2)])
def test_gpu_occupancy_matches_oracle(name, k):
    import torch

    import paper_2106_01326_b200 as pkg

    m = meshgen.make_config(name)
    if name == "cfg1":
        m = meshgen.carve_sphere(m)
    fine, g = _fine(m, k)
    off = m.tet_offsets if m.batch > 1 else None
    got_fine = pkg.voxelize(m.verts, m.tets, g, m.extent, tet_offsets=off)
    assert np.array_equal(got_fine, fine)
    d_fine = torch.from_numpy(got_fine.view(np.int32)).cuda()
    got = pkg.occupancy(d_fine, m.grid, k, batch=m.batch).cpu().numpy()
    exp = occupancy(fine, k)
    assert got.shape == exp.shape
    if not np.array_equal(got, exp):
        bad = np.argwhere(got != exp)
        raise AssertionError(f"{len(bad)} voxels differ, first {tuple(bad[0])}: gpu {got[tuple(bad[0])]} oracle {exp[tuple(bad[0])]}")


@pytest.mark.gpu
def test_gpu_occupancy_argument_checks():
    import ctypes

    import paper_2106_01326_b200 as pkg

    lib = pkg.load_library()
    p = ctypes.c_void_p(256)
    assert lib.vox_occupancy(None, p, 16, 4, 4, 1, 3, p) == -1      # k
    assert lib.vox_occupancy(None, p, 12, 4, 4, 1, 2, p) == -1      # (k*nx) % 32
    assert lib.vox_occupancy(None, None, 16, 4, 4, 1, 2, p) == -1


@pytest.mark.gpu
@pytest.mark.parametrize("nx,ny,nz,batch,k", [(16, 5, 3, 2, 4), (48, 7, 2, 1, 2), (64, 3, 5, 3, 2), (32, 4, 4, 1, 4),
                                               (8, 2, 2, 1, 4)])
def test_gpu_occupancy_on_random_bits(nx, ny, nz, batch, k):
    """Scalar and 16-byte-vector variants, odd row counts, batches: random fine bit grids straight into the fold."""
    import torch

    import paper_2106_01326_b200 as pkg

    rng = np.random.default_rng(nx * 131 + ny * 17 + nz + k)
    fine = rng.integers(0, 2**32, (batch, k * nz, k * ny, k * nx // 32), dtype=np.uint64).astype(np.uint32)
    fine[rng.random(fine.shape) < 0.2] = 0xFFFFFFFF
    got = pkg.occupancy(torch.from_numpy(fine.view(np.int32)).cuda(), (nx, ny, nz), k, batch=batch).cpu().numpy()
    assert np.array_equal(got, occupancy(fine, k))
