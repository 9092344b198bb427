"""Lattice input (include/vox.h "vox_lattice"): the same mesh given as lattice vertices + a keep
mask instead of a tet array must voxelize to the same bits as the oracle computes on the tets written out."""
import numpy as np
import pytest

import meshgen
import oracle
from meshgen.kuhn import Mesh, kuhn_mesh, _uniform_corners


def test_lattice_form_round_trips():
    m = meshgen.make_config("cfg2")
    keep = meshgen.lattice_form(m, (32, 32, 32))
    assert keep.dtype == np.uint8 and keep.shape == (32 ** 3,)
    assert int(np.unpackbits(keep).sum()) == m.T
    c = _uniform_corners(32)
    _v, t_all = kuhn_mesh(c, c, c, 0.0, None)           # connectivity only
    present = ((keep[:, None] >> np.arange(6)) & 1).astype(bool).reshape(-1)
    assert np.array_equal(t_all[present], m.tets)
    full = meshgen.make_config("cfg1")
    assert np.all(meshgen.lattice_form(full, (4, 4, 4)) == 63)


def _cases():
    rng = np.random.default_rng(44)
    out = []
    m = meshgen.carve_sphere(meshgen.make_config("cfg1"))
    out.append(("cfg1_sphere", m, (4, 4, 4)))
    out.append(("cfg2", meshgen.make_config("cfg2"), (32, 32, 32)))
    out.append(("cfg4_small_drop3", meshgen.carve_every_third(meshgen.make_config("cfg4_small")), (32, 32, 32)))
    # anisotropic lattice (different cell counts per axis), random carve, ragged grid
    xs, ys, zs = (np.rint(np.linspace(0, e, n + 1)).astype(np.int64) for e, n in ((96 * 8, 5), (40 * 8, 3), (24 * 8, 7)))
    v, t = kuhn_mesh(xs, ys, zs, 0.2, rng)
    t = t[rng.random(len(t)) < 0.6]
    out.append(("aniso", Mesh("aniso", v, t, (96, 40, 24), (96 * 8, 40 * 8, 24 * 8)), (5, 3, 7)))
    b = meshgen.make_config("cfg3_small")                    # a batch of 4 meshes on the same 24^3 lattice
    out.append(("cfg3_small", b, b.cells))
    # pitch 12 (not a power of two: the division forms of the box and the general plane setup), ragged grid
    xs, ys, zs = (np.rint(np.linspace(0, e, n + 1)).astype(np.int64) for e, n in ((64 * 12, 7), (40 * 12, 5), (24 * 12, 4)))
    v, t = kuhn_mesh(xs, ys, zs, 0.2, rng)
    t = t[rng.random(len(t)) < 0.7]
    out.append(("nonpow2", Mesh("nonpow2", v, t, (64, 40, 24), (64 * 12, 40 * 12, 24 * 12)), (7, 5, 4)))
    # sub-voxel cells: 40^3 cells on a 32^3 grid (0.8 voxel per cell): most tets hold no sample (culled per tile on
    # the fused path), a tile's index box holds tens of thousands of cells
    c = _uniform_corners(40)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    t = t[rng.random(len(t)) < 0.5]
    out.append(("subvoxel", Mesh("subvoxel", v, t, (32, 32, 32)), (40, 40, 40)))
    # giant cells: 2^3 cells on a 128^3 grid (every tile sees all 48 tets; int64 large path)
    g = meshgen.make_config("s1")
    out.append(("giant", Mesh("giant", g.verts, g.tets[::2].copy(), (128, 128, 128)), (2, 2, 2)))
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [2, 1], ids=["fused", "binned"])
@pytest.mark.parametrize("idx", range(8))
def test_gpu_lattice_input_matches_oracle(idx, variant):
    """variant 2: the fused lattice path (K0 slabs + tiles enumerating their own candidate cells, no K1-K3);
    variant 1: the same input through the binning passes.  Both must give the oracle's grid and count the same
    (tet, tile) pairs as the tet array written out."""
    import torch

    import paper_2106_01326_b200 as pkg

    name, m, cells = _cases()[idx]
    exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets)
    keep = meshgen.lattice_form(m, cells)
    vz = pkg.Voxelizer(m.grid, m.extent, m.batch, variant=variant)
    vz.set_lattice(torch.from_numpy(m.verts).cuda(), cells, torch.from_numpy(keep).cuda())
    assert vz.path == ("lattice_fused" if variant == 2 else "lattice_binned")
    if variant == 2:    # header + slabs + the 16-byte vertex copy: no counters, no range array, no pair list
        assert vz.workspace_bytes <= 1024 + 8 * m.batch * (sum(cells) + 3) + 16 * m.V + 768
    pairs = vz.plan()
    got = vz.run().cpu().numpy().view(np.uint32)
    st = vz.status()
    # sparse output through the same path
    from oracle import sparse
    ts = vz.tile_shape
    nb = m.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
    tab, pay = vz.run_sparse(nb)
    mixed = vz.sparse_status()["mixed_tiles"]
    vz.close()
    assert np.array_equal(got, exp), f"{name}: {(got != exp).sum()} words differ"
    assert sparse.check_table(tab.cpu().numpy(), pay.cpu().numpy(), exp, ts["ty"], ts["tz"]) == mixed
    # the same pairs as with the tets written out
    ref = pkg.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets if m.batch > 1 else None)
    assert np.array_equal(ref, exp) and pkg.voxelize.last_status["pairs"] == st["pairs"] == pairs
    assert pkg.voxelize.last_status["large_pairs"] == st["large_pairs"]


@pytest.mark.gpu
def test_gpu_default_path_of_lattice_input_and_launch_counts():
    """The default (variant 0) sends lattice input through the binning passes and picks the fused path by itself only
    for giant cells (mean cell >= 64^3 voxels); vox_path says which.  The launch counter (bench.py's gpu_launches)
    rises by exactly 4 per binned run (K1, K2, K3, K4) and by 2 per fused run (K0, K4)."""
    import torch

    import paper_2106_01326_b200 as pkg

    expect = {"cfg1_sphere": "lattice_binned", "cfg4_small_drop3": "lattice_binned", "giant": "lattice_fused"}
    seen = set()
    for name, m, cells in _cases():
        if name not in expect or m.batch > 1:
            continue
        seen.add(name)
        exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
        keep = meshgen.lattice_form(m, cells)
        dv, dk = torch.from_numpy(m.verts).cuda(), torch.from_numpy(keep).cuda()
        for variant, path in ((0, expect[name]), (1, "lattice_binned"), (2, "lattice_fused")):
            vz = pkg.Voxelizer(m.grid, m.extent, 1, variant=variant)
            vz.set_lattice(dv, cells, dk)
            assert vz.path == path, (name, variant, vz.path)
            vz.plan()
            out = vz.run()
            torch.cuda.synchronize()
            before = pkg.kernel_launches()
            for _ in range(3):
                vz.run(out)
            assert pkg.kernel_launches() - before == 3 * (2 if path == "lattice_fused" else 4), (name, variant)
            assert np.array_equal(out.cpu().numpy().view(np.uint32), exp), (name, variant)
            vz.close()
        # the tet array: path 'tets', 4 launches
        vz = pkg.Voxelizer(m.grid, m.extent, 1)
        vz.set_tets(dv, torch.from_numpy(m.tets).cuda())
        assert vz.path == "tets"
        vz.plan()
        out = vz.run()
        before = pkg.kernel_launches()
        vz.run(out)
        assert pkg.kernel_launches() - before == 4
        vz.close()
    assert seen == set(expect)


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [0, 2], ids=["default", "fused"])
def test_gpu_lattice_through_the_pipe_dense_and_sparse(variant):
    import torch

    import paper_2106_01326_b200 as pkg
    from oracle import sparse

    name, m, cells = _cases()[1]
    exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
    keep = meshgen.lattice_form(m, cells)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    pipe = pkg.Pipe(m.grid, m.extent, depth=3, max_V=m.V, max_T=6 * cells[0] * cells[1] * cells[2], variant=variant)
    ts = pipe.tile_shape
    nb = ts["nbx"] * ts["nby"] * ts["nbz"]
    nx, ny, nz = m.grid
    h_out = torch.empty((1, nz, ny, nx // 32), dtype=torch.int32).pin_memory()
    h_tab = torch.zeros(nb, dtype=torch.int32).pin_memory()
    h_pay = torch.zeros((nb, ts["tz"], ts["ty"]), dtype=torch.int32).pin_memory()
    t0 = pipe.submit_lattice(pin(m.verts), cells, pin(keep), h_out)
    t1 = pipe.submit_lattice(pin(m.verts), cells, pin(keep), h_tab, h_pay, nb)
    t2 = pipe.submit(pin(m.verts), pin(m.tets), h_out.clone().pin_memory())     # explicit tets after a lattice job
    pipe.wait(t0)
    st = pipe.wait(t1)
    pipe.wait(t2)
    pipe.close()
    assert np.array_equal(h_out.numpy().view(np.uint32), exp)
    assert sparse.check_table(h_tab.numpy(), h_pay.numpy(), exp, ts["ty"], ts["tz"]) == st["mixed_tiles"]


@pytest.mark.gpu
def test_gpu_batched_lattice_through_the_pipe():
    import torch

    import paper_2106_01326_b200 as pkg

    m = meshgen.make_config("cfg3_small")
    exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets)
    keep = meshgen.lattice_form(m, m.cells)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    pipe = pkg.Pipe(m.grid, m.extent, m.batch, depth=2, max_V=m.V, max_T=m.batch * 6 * 24 ** 3)
    nx, ny, nz = m.grid
    outs = [torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32).pin_memory() for _ in range(2)]
    ts = [pipe.submit_lattice(pin(m.verts), m.cells, pin(keep), o) for o in outs]
    for t in ts:
        pipe.wait(t)
    pipe.close()
    for o in outs:
        assert np.array_equal(o.numpy().view(np.uint32), exp)


@pytest.mark.gpu
@pytest.mark.parametrize("block", range(4))
def test_gpu_random_lattices_match_oracle(block):
    """Random background lattices: 1..13 cells per axis (from one giant cell per tile row to cells of a few lattice
    units), jitter 0..0.3 cell, 20..100 % of the tets kept, ragged grids with power-of-two and other pitches -- through
    the fused path and through the binning passes, each against the oracle on the tets written out.
    (Round-2 soaks of 10 000 random tet jobs and 2 500 such lattices, both lattice paths, ran without a differing word; this keeps 48 lattices in the suite.)"""
    import torch

    import paper_2106_01326_b200 as pkg

    done = 0
    for seed in range(12 * block, 12 * (block + 1)):
        rng = np.random.default_rng(50000 + seed)
        cells = tuple(int(rng.integers(1, 14)) for _ in range(3))
        n = (32 * int(rng.integers(1, 4)), int(rng.integers(4, 60)), int(rng.integers(4, 60)))
        pitch = [2 * int(rng.integers(1, 40)) for _ in range(3)] if seed % 2 else [int(2 ** rng.integers(1, 8))] * 3
        ext = tuple(a * b for a, b in zip(n, pitch))
        cs = [np.rint(np.linspace(0, e, c + 1)).astype(np.int64) for e, c in zip(ext, cells)]
        if any(np.any(np.diff(c) < 1) for c in cs):
            continue
        v, t = kuhn_mesh(cs[0], cs[1], cs[2], float(rng.uniform(0, 0.3)), rng)
        t = t[rng.random(len(t)) < rng.uniform(0.2, 1.0)]
        m = Mesh(f"lat{seed}", v, t, n, ext)
        exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
        keep = meshgen.lattice_form(m, cells)
        pairs = []
        for variant in (2, 1):
            vz = pkg.Voxelizer(m.grid, m.extent, 1, variant=variant)
            vz.set_lattice(torch.from_numpy(m.verts).cuda(), cells, torch.from_numpy(keep).cuda())
            vz.plan()
            got = vz.run().cpu().numpy().view(np.uint32)
            pairs.append(vz.status()["pairs"])
            vz.close()
            assert np.array_equal(got, exp), f"seed {seed} cells {cells} grid {n} extent {ext} variant {variant}: {(got != exp).sum()} words differ"
        assert pairs[0] == pairs[1], (seed, pairs)
        done += 1
    assert done >= 8


@pytest.mark.gpu
def test_gpu_fused_lattice_with_a_huge_index_box():
    """160^3 sub-voxel cells on a 32^3 grid with one 32^3 tile: the tile's index box holds 4.1 M cells, beyond the 2^21
    up to which the fused path decodes a cell with float reciprocals -- the integer-division branch of the
    enumeration.  8 % of the tets kept; nearly all of them hold no sample and are skipped per tile."""
    import torch

    import paper_2106_01326_b200 as pkg

    rng = np.random.default_rng(99)
    C = 160
    c = _uniform_corners(C)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    t = t[rng.random(len(t)) < 0.08]
    m = Mesh("hugebox", v, t, (32, 32, 32))
    exp = oracle.voxelize(m.verts, m.tets, m.grid, m.extent)
    keep = meshgen.lattice_form(m, (C, C, C))
    dv, dk = torch.from_numpy(m.verts).cuda(), torch.from_numpy(keep).cuda()
    pairs = {}
    for tile in ((32, 32), (8, 8)):
        for variant in (2, 1):
            vz = pkg.Voxelizer(m.grid, m.extent, 1, tile=tile, variant=variant)
            vz.set_lattice(dv, (C, C, C), dk)
            vz.plan()
            got = vz.run().cpu().numpy().view(np.uint32)
            pairs[(tile, variant)] = vz.status()["pairs"]
            vz.close()
            assert np.array_equal(got, exp), f"tile {tile} variant {variant}: {(got != exp).sum()} words differ"
        assert pairs[(tile, 2)] == pairs[(tile, 1)] > 0
