"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, bit for bit.

Integer work: the bar is bit-exact equality of the whole grid."""
import numpy as np
import pytest

import meshgen
import oracle
from meshgen.kuhn import Mesh, kuhn_mesh

pytestmark = pytest.mark.gpu
E = 65536


def gpu_voxelize(m, **kw):
    import paper_2106_01326_b200 as pkg

    off = m.tet_offsets if m.batch > 1 else None
    return pkg.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=off, **kw)


def cpu_voxelize(m):
    return oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets)


def assert_same(got, exp, what=""):
    if not np.array_equal(got, exp):
        bad = np.argwhere(got != exp)
        b = tuple(bad[0])
        raise AssertionError(
            f"{what}: {len(bad)} differing words; first at [m,z,y,xw]={b}: gpu={got[b]:#010x} oracle={exp[b]:#010x}; "
            f"popcount gpu={int(np.unpackbits(got.view(np.uint8)).sum())} oracle={int(np.unpackbits(exp.view(np.uint8)).sum())}"
        )


def test_p1_single_tet():
    m = meshgen.single_tet_mesh((0, 0, 0), (8192, 0, 0), (8192, 8192, 0), (8192, 8192, 8192))
    got = gpu_voxelize(m)
    assert_same(got, cpu_voxelize(m), "p1")
    assert int(np.unpackbits(got.view(np.uint8)).sum()) == 20


def _giant(grid=256, jitter=0.2, seed=1101):
    m = meshgen.make_config("s1", seed)
    if jitter == 0.0:
        c = np.array([0, E // 2, E])
        v, t = kuhn_mesh(c, c, c, 0.0, None)
        m = Mesh("s1_nojit", v, t, (grid,) * 3, expect_all_ones=True)
    return Mesh(m.name + f"_{grid}", m.verts, m.tets, (grid,) * 3, expect_all_ones=True)


CASES = {
    "cfg1": lambda: meshgen.make_config("cfg1"),
    "cfg1_drop3": lambda: meshgen.carve_every_third(meshgen.make_config("cfg1")),
    "cfg1_sphere": lambda: meshgen.carve_sphere(meshgen.make_config("cfg1")),
    "cfg2": lambda: meshgen.make_config("cfg2"),
    "cfg2_drop3": lambda: meshgen.carve_every_third(meshgen.make_config("cfg2")),
    "cfg3_small": lambda: meshgen.make_config("cfg3_small"),
    "cfg4_small": lambda: meshgen.make_config("cfg4_small"),
    "cfg4_small_drop3": lambda: meshgen.carve_every_third(meshgen.make_config("cfg4_small")),
    "giant256": lambda: _giant(256),
    "giant256_nojit": lambda: _giant(256, 0.0),
    "giant256_drop3": lambda: meshgen.carve_every_third(_giant(256)),
    "giant128_sphere": lambda: meshgen.carve_sphere(_giant(128), 0.45),
}


@pytest.mark.parametrize("name", list(CASES))
def test_parity_small_configs(name):
    m = CASES[name]()
    exp = cpu_voxelize(m)
    got = gpu_voxelize(m)
    assert_same(got, exp, name)
    if m.expect_all_ones:
        assert np.all(got == np.uint32(0xFFFFFFFF))


@pytest.mark.parametrize("name", ["cfg3", "cfg4", "cfg5"])
def test_parity_full_size_configs(name):
    """BASELINE.json's full sizes in the launch configuration bench.py times (default tile and
    variant, vox_plan for the workspace): the whole grid against the oracle, which finishes each
    of these in seconds (3.4e9 candidate samples at cfg4)."""
    m = meshgen.make_config(name)
    exp = cpu_voxelize(m)
    got = gpu_voxelize(m)
    assert_same(got, exp, name + " full size")
    if m.expect_all_ones:
        assert np.all(got == np.uint32(0xFFFFFFFF))


@pytest.mark.parametrize("tile", [(32, 32), (8, 8), (16, 4), (4, 32), (32, 4)])
@pytest.mark.parametrize("name", ["cfg2", "cfg4_small_drop3", "giant128_sphere"])
def test_parity_is_tile_independent(name, tile):
    m = CASES[name]()
    assert_same(gpu_voxelize(m, tile=tile), cpu_voxelize(m), f"{name} tile={tile}")


def test_unknown_kernel_variant_is_refused():
    # variants 0 (default), 1 (binned lattice path) and 2 (fused lattice path) exist; any other must be refused
    import paper_2106_01326_b200 as pkg

    with pytest.raises(pkg.VoxError) as ei:
        pkg.Voxelizer((32, 32, 32), variant=3)
    assert ei.value.code == -1
    with pytest.raises(pkg.VoxError):
        pkg.Pipe((32, 32, 32), depth=1, max_V=4, max_T=1, variant=4)


def test_graph_replay_of_a_step_matches_oracle():
    """vox_run only enqueues, so a step can be captured into a CUDA graph and replayed (Voxelizer.capture)."""
    import torch

    import paper_2106_01326_b200 as pkg

    for name in ("cfg2", "cfg3_small"):
        m = CASES[name]()
        exp = cpu_voxelize(m)
        vz = pkg.Voxelizer(m.grid, m.extent, m.batch)
        off = torch.from_numpy(m.tet_offsets).cuda() if m.batch > 1 else None
        vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda(), off)
        vz.plan()
        nx, ny, nz = m.grid
        out = torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32, device="cuda")
        g = vz.capture(out, steps=2)
        for _ in range(3):
            out.fill_(-1)                      # stale bits must be overwritten by every replay
            g.replay()
            torch.cuda.synchronize()
            assert_same(out.cpu().numpy().view(np.uint32), exp, f"graph replay {name}")
        assert vz.status()["pairs"] > 0
        vz.close()


def test_graph_capture_skips_timing_events_and_refuses_a_rebound_voxelizer():
    """With vox_timing_enable active a captured vox_run records no events and takes no run number (the events of the
    runs outside the capture stay readable); a CapturedStep refuses to replay once the Voxelizer's workspace or mesh
    has been re-bound, because the graph still holds the old pointers."""
    import torch

    import paper_2106_01326_b200 as pkg

    m = CASES["cfg2"]()
    exp = cpu_voxelize(m)
    vz = pkg.Voxelizer(m.grid, m.extent, m.batch)
    vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda())
    vz.plan()
    vz.timing_enable(8)
    nx, ny, nz = m.grid
    out = torch.empty((1, nz, ny, nx // 32), dtype=torch.int32, device="cuda")
    vz.run(out)                      # run 0
    g = vz.capture(out, steps=2)     # its warm-up outside the capture is run 1; the two captured runs take no number
    torch.cuda.synchronize()
    for run in (0, 1):
        ms = vz.timing_read(run)
        assert ms["total"] > 0 and ms["k4"] > 0
    with pytest.raises(pkg.VoxError) as ei:
        vz.timing_read(2)
    assert ei.value.code == -5
    for _ in range(2):
        out.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        assert_same(out.cpu().numpy().view(np.uint32), exp, "graph replay with timing enabled")
    assert vz.timing_read(1)["total"] > 0     # replays did not disturb the ring
    vz.run(out)                                # run 2, outside any capture
    torch.cuda.synchronize()
    assert vz.timing_read(2)["total"] > 0
    vz.alloc_workspace()                       # re-binds the workspace: the graph's pointer is stale
    with pytest.raises(RuntimeError):
        g.replay()
    vz.close()


def test_estimated_workspace_path():
    m = CASES["cfg2"]()
    assert_same(gpu_voxelize(m, exact_plan=False), cpu_voxelize(m), "cfg2 without vox_plan")


def test_host_buffer_entry_point():
    import paper_2106_01326_b200 as pkg

    for name in ["cfg2", "cfg3_small"]:
        m = CASES[name]()
        off = m.tet_offsets if m.batch > 1 else None
        got = pkg.voxelize_host(m.verts, m.tets, m.grid, m.extent, tet_offsets=off)
        assert_same(got, cpu_voxelize(m), name + " via vox_run_host")


# ------------------------------------------------------------------ edge cases
def test_empty_mesh_gives_zero_grid():
    m = Mesh("empty", np.zeros((4, 3), np.int32), np.zeros((0, 4), np.int32), (64, 32, 32))
    got = gpu_voxelize(m)
    assert got.shape == (1, 32, 32, 2) and not got.any()


def test_all_tets_culled():
    # degenerate (coplanar, repeated vertex) and sub-voxel slivers between sample planes
    v = np.array([[0, 0, 1024], [E, 0, 1024], [0, E, 1024], [E, E, 1024],
                  [10, 10, 10], [500, 10, 10], [10, 500, 10], [10, 10, 500]], dtype=np.int32)
    t = np.array([[0, 1, 2, 3], [0, 1, 2, 2], [1, 1, 1, 1], [4, 5, 6, 7]], dtype=np.int32)
    m = Mesh("culled", v, t, (32, 32, 32))
    got = gpu_voxelize(m)
    assert not got.any() and not cpu_voxelize(m).any()
    import paper_2106_01326_b200 as pkg

    assert pkg.voxelize.last_status["culled"] == 4 and pkg.voxelize.last_status["pairs"] == 0


def test_stale_output_is_overwritten():
    import torch

    import paper_2106_01326_b200 as pkg

    m = CASES["cfg1_sphere"]()
    vz = pkg.Voxelizer(m.grid)
    vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda())
    out = torch.full((1, 32, 32, 1), -1, dtype=torch.int32, device="cuda")
    vz.plan()
    vz.run(out)
    vz.run(out)  # twice into the same buffers: no stale state in the workspace either
    vz.status()
    assert_same(out.cpu().numpy().view(np.uint32), cpu_voxelize(m), "rerun")
    vz.close()


@pytest.mark.parametrize(
    "grid,extent",
    [((32, 24, 40), (32 * 6, 24 * 10, 40 * 14)),     # pitches 6,10,14: gcd 2
     ((64, 20, 12), (64 * 6, 20 * 12, 12 * 18)),     # pitches 6,12,18: gcd 6 (not a power of two)
     ((32, 40, 24), (32 * 2048, 40 * 512, 24 * 4096)),
     ((96, 33, 7), (96 * 4, 33 * 4, 7 * 4)),
     ((4096, 40, 24), (4096 * 16, 40 * 512, 24 * 1024))],   # 128 tiles along x
)
def test_ragged_anisotropic_grids(grid, extent):
    rng = np.random.default_rng(sum(grid))
    cs = [np.rint(np.linspace(0, extent[k], 4 + k)).astype(np.int64) for k in range(3)]
    v, t = kuhn_mesh(cs[0], cs[1], cs[2], 0.2, rng)
    # move boundary vertices too (kept inside the box), then carve
    v = np.clip(v + rng.integers(-2, 3, v.shape), 0, np.array(extent)).astype(np.int32)
    t = t[rng.random(len(t)) < 0.7]
    m = Mesh("ragged", v, t, grid, extent)
    exp = cpu_voxelize(m)
    assert exp.any() and not np.all(exp == np.uint32(0xFFFFFFFF))
    for tile in [None, (4, 4), (16, 8)]:
        assert_same(gpu_voxelize(m, tile=tile), exp, f"ragged {grid} tile={tile}")


def test_max_extent_forces_the_int64_large_path():
    # extent 2^20: plane coefficients exceed int32 on every tile
    Emax = 1 << 20
    rng = np.random.default_rng(5)
    c = np.rint(np.linspace(0, Emax, 4)).astype(np.int64)
    v, t = kuhn_mesh(c, c, c, 0.2, rng)
    t = t[rng.random(len(t)) < 0.6]
    m = Mesh("emax", v, t, (64, 64, 64), (Emax,) * 3)
    got = gpu_voxelize(m)
    assert_same(got, cpu_voxelize(m), "extent 2^20")
    import paper_2106_01326_b200 as pkg

    assert pkg.voxelize.last_status["large_pairs"] > 0


def test_random_soup_with_overlaps_and_inverted_tets():
    # not a conforming mesh: random tets of all sizes, both orientations, overlapping
    rng = np.random.default_rng(77)
    v = rng.integers(0, E + 1, (400, 3)).astype(np.int32)
    t = np.array([rng.choice(400, 4, replace=False) for _ in range(300)], dtype=np.int32)
    small = (v[:200] // 16 + 30000).astype(np.int32)  # a cluster of small tets
    v[:200] = small
    m = Mesh("soup", v, t, (64, 64, 64))
    assert_same(gpu_voxelize(m), cpu_voxelize(m), "soup")


def test_vertices_on_sample_points_and_faces():
    # coordinates on multiples of h/2: samples exactly on faces, edges and vertices (inclusive test)
    rng = np.random.default_rng(61)
    h = 2048
    pts = (rng.integers(0, 65, (60, 3)) * (h // 2)).astype(np.int32)
    t = np.array([rng.choice(60, 4, replace=False) for _ in range(120)], dtype=np.int32)
    m = Mesh("onfaces", pts, t, (32, 32, 32))
    assert_same(gpu_voxelize(m), cpu_voxelize(m), "on-faces")
    h = 512
    pts = (rng.integers(40, 90, (80, 3)) * (h // 2)).astype(np.int32)  # small tets: int32 fast path
    t = np.array([rng.choice(80, 4, replace=False) for _ in range(200)], dtype=np.int32)
    m = Mesh("onfaces_small", pts, t, (128, 128, 128))
    assert_same(gpu_voxelize(m), cpu_voxelize(m), "on-faces small")


def test_workspace_overflow_is_reported():
    import torch

    import paper_2106_01326_b200 as pkg

    m = CASES["cfg2"]()
    vz = pkg.Voxelizer(m.grid)
    vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda())
    vz.alloc_workspace(vz.workspace_fixed_bytes + 4096)  # room for 1024 pairs only
    vz.run()
    with pytest.raises(pkg.VoxError) as ei:
        vz.status()
    assert ei.value.code == -3
    pairs = vz.plan()
    assert pairs > 1024
    vz.run()
    assert vz.status()["pairs"] == pairs
    vz.close()


def test_validate_flags_bad_data():
    import torch

    import paper_2106_01326_b200 as pkg

    m = CASES["cfg1"]()
    vz = pkg.Voxelizer(m.grid)
    v = torch.from_numpy(m.verts).cuda()
    t = torch.from_numpy(m.tets).cuda()
    vz.set_tets(v, t)
    vz.validate()
    t2 = t.clone()
    t2[5, 2] = m.V
    vz.set_tets(v, t2)
    with pytest.raises(pkg.VoxError) as ei:
        vz.validate()
    assert ei.value.code == -6
    v2 = v.clone()
    v2[3, 1] = E + 1
    vz.set_tets(v2, t)
    with pytest.raises(pkg.VoxError):
        vz.validate()
    vz.close()


# ------------------------------------------------------------------ vox_pipe
def _pinned(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


def test_pipe_stream_of_meshes_matches_oracle():
    """Seven different meshes through a depth-3 pipeline (slots are reused, in-flight overlap):
    every grid must equal the oracle's, bit for bit, and the stats must be per mesh."""
    import torch

    import paper_2106_01326_b200 as pkg

    base = meshgen.make_config("cfg2")
    meshes = [base, meshgen.carve_every_third(base), meshgen.carve_sphere(base, 0.3)]
    for seed in (11, 12, 13):
        meshes.append(meshgen.make_config("cfg2", seed))
    meshes.append(Mesh("empty", base.verts, base.tets[:0], base.grid))
    pipe = pkg.Pipe(base.grid, depth=3, max_V=max(m.V for m in meshes), max_T=max(m.T for m in meshes))
    nx, ny, nz = base.grid
    outs = [torch.full((1, nz, ny, nx // 32), -1, dtype=torch.int32).pin_memory() for _ in meshes]
    tickets = [pipe.submit(_pinned(m.verts), _pinned(m.tets), o) for m, o in zip(meshes[:3], outs[:3])]
    stats = {}
    for k in range(3, len(meshes)):          # keep three in flight
        stats[tickets[k - 3]] = pipe.wait(tickets[k - 3])
        tickets.append(pipe.submit(_pinned(meshes[k].verts), _pinned(meshes[k].tets), outs[k]))
    for t in tickets[-3:]:
        stats[t] = pipe.wait(t)
    assert tickets == list(range(len(meshes)))
    for k, (m, o) in enumerate(zip(meshes, outs)):
        assert_same(o.numpy().view(np.uint32), cpu_voxelize(m), f"pipe mesh {k} ({m.name})")
    assert stats[len(meshes) - 1]["pairs"] == 0 and stats[0]["pairs"] > 0
    with pytest.raises(pkg.VoxError) as ei:   # a ticket can be waited on once
        pipe.wait(0)
    assert ei.value.code == -5
    pipe.close()


def test_pipe_batched_meshes_and_limits():
    import torch

    import paper_2106_01326_b200 as pkg

    m = meshgen.make_config("cfg3_small")
    pipe = pkg.Pipe(m.grid, batch=m.batch, depth=2, max_V=m.V, max_T=m.T)
    nx, ny, nz = m.grid
    exp = cpu_voxelize(m)
    outs = [torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32).pin_memory() for _ in range(4)]
    hv, ht, ho = _pinned(m.verts), _pinned(m.tets), _pinned(m.tet_offsets)
    ts = [pipe.submit(hv, ht, o, ho) for o in outs]   # 4 submits into 2 slots: submit blocks on the oldest
    for t in ts[2:]:
        pipe.wait(t)
    for o in outs:
        assert_same(o.numpy().view(np.uint32), exp, "pipe batched")
    big = torch.zeros((m.T + 1, 4), dtype=torch.int32).pin_memory()
    with pytest.raises(pkg.VoxError) as ei:
        pipe.submit(hv, big, outs[0], ho)
    assert ei.value.code == -2
    pipe.close()


# ------------------------------------------------------------------ sparse output
def _gpu_sparse(m, tile=None, capacity=None):
    import torch

    import paper_2106_01326_b200 as pkg

    off = torch.from_numpy(m.tet_offsets).cuda() if m.batch > 1 else None
    vz = pkg.Voxelizer(m.grid, m.extent, m.batch, tile=tile)
    try:
        vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda(), off)
        vz.plan()
        ts = vz.tile_shape
        nb = m.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
        cap = nb if capacity is None else capacity
        table, payload = vz.run_sparse(cap)
        st = vz.sparse_status()
        return table.cpu().numpy().view(np.uint32), payload.cpu().numpy().view(np.uint32), ts, st
    finally:
        vz.close()


@pytest.mark.parametrize("name,tile", [("cfg1_sphere", None), ("cfg2", None), ("cfg2", (8, 8)), ("cfg3_small", None),
                                       ("cfg4_small_drop3", None), ("giant128_sphere", (16, 4)), ("cfg5", None)])
def test_sparse_output_matches_oracle(name, tile):
    from oracle import sparse

    m = CASES[name]() if name in CASES else meshgen.make_config(name)
    exp = cpu_voxelize(m)
    table, payload, ts, st = _gpu_sparse(m, tile)
    mixed = sparse.check_table(table, payload, exp, ts["ty"], ts["tz"])   # classes, slots, payload content
    assert st["mixed_tiles"] == mixed
    assert st["full_tiles"] == int(np.sum(table == np.uint32(0xFFFFFFFF)))
    assert_same(sparse.decode(table, payload, m.grid, m.batch, ts["ty"], ts["tz"]), exp, name + " sparse decode")


def test_sparse_ragged_grid_and_capacity_overflow():
    import paper_2106_01326_b200 as pkg
    from oracle import sparse

    rng = np.random.default_rng(9)
    grid, extent = (64, 20, 12), (64 * 6, 20 * 12, 12 * 18)
    cs = [np.rint(np.linspace(0, extent[k], 4 + k)).astype(np.int64) for k in range(3)]
    v, t = kuhn_mesh(cs[0], cs[1], cs[2], 0.2, rng)
    t = t[rng.random(len(t)) < 0.8]
    m = Mesh("ragged_sparse", v, t, grid, extent)
    exp = cpu_voxelize(m)
    for tile in [(8, 8), (16, 8), (32, 32)]:
        table, payload, ts, st = _gpu_sparse(m, tile)
        assert sparse.check_table(table, payload, exp, ts["ty"], ts["tz"]) == st["mixed_tiles"] > 0
    with pytest.raises(pkg.VoxError) as ei:      # room for one payload tile only
        _gpu_sparse(m, (8, 8), capacity=1)
    assert ei.value.code == -3


def test_pipe_sparse_payload_lands_in_pinned_host_memory():
    import torch

    import paper_2106_01326_b200 as pkg
    from oracle import sparse

    base = meshgen.make_config("cfg2")
    meshes = [base, meshgen.carve_every_third(base), meshgen.make_config("cfg2", 21), meshgen.carve_sphere(base, 0.3)]
    pipe = pkg.Pipe(base.grid, depth=2, max_V=max(m.V for m in meshes), max_T=max(m.T for m in meshes))
    ts = pipe.tile_shape
    nb = ts["nbx"] * ts["nby"] * ts["nbz"]
    tables = [torch.zeros(nb, dtype=torch.int32).pin_memory() for _ in meshes]
    pays = [torch.zeros((nb, ts["tz"], ts["ty"]), dtype=torch.int32).pin_memory() for _ in meshes]
    tickets, stats = [], []
    for k, m in enumerate(meshes):
        if k >= 2:
            stats.append(pipe.wait(tickets[k - 2]))
        tickets.append(pipe.submit_sparse(_pinned(m.verts), _pinned(m.tets), tables[k], pays[k], nb))
    stats += [pipe.wait(t) for t in tickets[-2:]]
    for k, m in enumerate(meshes):
        exp = cpu_voxelize(m)
        tb, pl = tables[k].numpy().view(np.uint32), pays[k].numpy().view(np.uint32)
        assert sparse.check_table(tb, pl, exp, ts["ty"], ts["tz"]) == stats[k]["mixed_tiles"]
        assert_same(sparse.decode(tb, pl, m.grid, 1, ts["ty"], ts["tz"]), exp, f"pipe sparse {k}")
    pipe.close()


def test_planes_with_unit_and_zero_x_normal_component():
    """Faces whose normal has x-component 0, +-1 or +-2 (the reciprocal's corner cases: |mx| = 1 is stored
    scaled by 4, mx = 0 only gates the row).  Includes the tet that exposed a ptxas folding of `mx == -1`."""
    rng = np.random.default_rng(2126)
    verts = [[13118, 38472, 44237], [13629, 37852, 46741], [13779, 40783, 46370], [16778, 40704, 46380]]
    tets = [[0, 1, 2, 3]]
    for i in range(300):
        a = rng.integers(6000, 50000, 3)
        p, q = int(rng.integers(800, 4000)), int(rng.integers(-4000, 4000))
        k = int(rng.integers(-3, 4))
        c = int(rng.integers(0, 3))               # x-component of u x v = c  (u = (p,c,0), v = (q,k,1))
        u, v = np.array([p, c, 0]), np.array([q, k, 1])
        if i % 3 == 1:
            u, v = v, u                           # -> x-component = -c
        d = rng.integers(-6000, 6000, 3)
        base = len(verts)
        verts += [a.tolist(), (a + u).tolist(), (a + v).tolist(), (a + d).tolist()]
        tets.append([base, base + 1, base + 2, base + 3])
    m = Mesh("unit_nx", np.array(verts, dtype=np.int32), np.array(tets, dtype=np.int32), (64, 64, 64))
    exp = cpu_voxelize(m)
    assert exp.any()
    for tile in [None, (32, 32), (8, 8)]:
        assert_same(gpu_voxelize(m, tile=tile), exp, f"unit nx tile={tile}")
    m2 = Mesh("unit_nx_fine", m.verts, m.tets, (256, 256, 256))
    assert_same(gpu_voxelize(m2), cpu_voxelize(m2), "unit nx 256^3")


# ------------------------------------------------------------------ randomized differential test
def _random_job(seed):
    """A random grid (anisotropic pitches, ragged dims), a random batch and a soup of tets of every size class:
    sub-voxel slivers, few-voxel tets, tile-sized tets, grid-spanning giants, degenerate and axis-aligned ones."""
    rng = np.random.default_rng(seed)
    nx = 32 * int(rng.integers(1, 5))
    ny, nz = int(rng.integers(1, 71)), int(rng.integers(1, 71))
    pitch = [2 * int(rng.integers(1, 600)) for _ in range(3)]
    if seed % 3 == 0:
        pitch = [int(2 ** rng.integers(1, 11))] * 3          # the common case: equal power-of-two pitches
    extent = (nx * pitch[0], ny * pitch[1], nz * pitch[2])
    if max(extent) > (1 << 20):
        return None
    batch = int(rng.integers(1, 4))
    ext = np.array(extent)
    verts, tets, offsets = [], [], [0]
    for _ in range(batch):
        n_t = int(rng.integers(0, 120))
        for _t in range(n_t):
            kind = rng.integers(0, 6)
            c = rng.integers(0, ext + 1)
            size = [np.array(pitch) // 2 + 1, np.array(pitch) * 3, np.array(pitch) * 12, ext // 2 + 1, ext + 1,
                    np.array(pitch) * 3][kind]
            pts = c + rng.integers(-size, size + 1, (4, 3))
            if kind == 5:                                      # axis-aligned faces / samples on faces
                pts = (pts // (np.array(pitch) // 2 + 1)) * (np.array(pitch) // 2 + 1)
            if rng.random() < 0.05:
                pts[3] = pts[rng.integers(0, 3)]               # degenerate: repeated vertex
            pts = np.clip(pts, 0, ext)
            base = len(verts)
            verts += pts.tolist()
            tets.append([base, base + 1, base + 2, base + 3])
        offsets.append(len(tets))
    if not verts:
        verts = [[0, 0, 0]] * 4
    v = np.array(verts, dtype=np.int32).reshape(-1, 3)
    t = np.array(tets, dtype=np.int32).reshape(-1, 4)
    m = Mesh(f"fuzz{seed}", v, t, (nx, ny, nz), extent)
    if batch > 1:
        m = Mesh(f"fuzz{seed}", v, t, (nx, ny, nz), extent, tet_offsets=np.array(offsets, dtype=np.int64))
    tile = [None, (4, 4), (8, 32), (32, 32), (16, 8)][int(rng.integers(0, 5))]
    return m, tile


@pytest.mark.parametrize("block", range(6))
def test_randomized_jobs_match_oracle(block):
    from oracle import sparse

    done = 0
    for seed in range(1000 + 12 * block, 1000 + 12 * (block + 1)):
        job = _random_job(seed)
        if job is None:
            continue
        m, tile = job
        exp = cpu_voxelize(m)
        got = gpu_voxelize(m, tile=tile)
        assert_same(got, exp, f"fuzz seed {seed} grid {m.grid} extent {m.extent} batch {m.batch} tile {tile}")
        if seed % 4 == 0:
            table, payload, ts, st = _gpu_sparse(m, tile)
            assert sparse.check_table(table, payload, exp, ts["ty"], ts["tz"]) == st["mixed_tiles"], f"seed {seed}"
        done += 1
    assert done >= 6


def test_randomized_magnitudes_straddle_the_int32_limit():
    """Random tets of 2^4..2^14.5 lattice units on lattices of extent 2^14..2^20: a good part of the (tet, tile)
    pairs fits the int32 span path and a good part takes the int64 large path (plane values beyond int32, or bbox
    extents beyond 2^15), so the hand-over bound is exercised from both sides."""
    import paper_2106_01326_b200 as pkg

    large = pairs = 0
    for seed in range(80):
        rng = np.random.default_rng(seed)
        n = int(rng.choice([32, 64, 128, 256]))
        Ex = 1 << int(rng.integers(14, 21))
        verts, tets = [], []
        for _ in range(int(rng.integers(5, 60))):
            size = int(2 ** rng.uniform(4, 14.5))
            c = rng.integers(0, Ex + 1, 3)
            pts = np.clip(c + rng.integers(-size // 2, size // 2 + 1, (4, 3)), 0, Ex)
            b = len(verts)
            verts += pts.tolist()
            tets.append([b, b + 1, b + 2, b + 3])
        m = Mesh(f"mag{seed}", np.array(verts, dtype=np.int32), np.array(tets, dtype=np.int32), (n, n, n), (Ex,) * 3)
        tile = [None, (8, 8), (32, 32)][int(rng.integers(0, 3))]
        assert_same(gpu_voxelize(m, tile=tile), cpu_voxelize(m), f"magnitude seed {seed} n {n} E {Ex} tile {tile}")
        large += pkg.voxelize.last_status["large_pairs"]
        pairs += pkg.voxelize.last_status["pairs"]
    print(f"straddle: large={large} span={pairs - large} pairs={pairs}")
    # fixed seeds: explicit floors on BOTH sides of the hand-over (measured at round 3: see the printed line with -s)
    assert large >= STRADDLE_MIN_LARGE and pairs - large >= STRADDLE_MIN_SPAN, (large, pairs)


# measured with these seeds at round 3: 11 941 pairs on the int64 path, 5 009 on the int32 span path (of 16 950).  A change
# that moves the hand-over may move these by a little; one that pushes either side below the floor has stopped
# exercising that side and must say so by changing the floor.
STRADDLE_MIN_LARGE = 10000
STRADDLE_MIN_SPAN = 4000


def test_single_tet_swept_across_the_int32_hand_over():
    """One tet shape grown in 2 % steps from 2^12 to 2^15.4 lattice units on a 256^3 grid of extent 2^20 (pitch 4096):
    the int32 span record holds it at the small end (plane values ~ d^3 / g below 2^31) and cannot at the large end, so
    the sweep crosses the hand-over bound with neighbours 2 % apart on either side of it -- every grid against the
    oracle, on two tile shapes, and both ends must be on the side they belong to."""
    import paper_2106_01326_b200 as pkg

    Ex, n = 1 << 20, 256
    base = np.array([300000, 410000, 520000])
    shape = np.array([[0.0, 0.0, 0.0], [1.0, 0.13, 0.21], [0.17, 0.93, 0.08], [0.22, 0.31, 0.97]])
    for tile in ((32, 32), (8, 8)):
        flags = []
        for k in range(120):
            d = 4096.0 * 1.02 ** k
            pts = np.clip(np.rint(base + shape * d).astype(np.int64), 0, Ex)
            m = Mesh(f"sweep{k}", pts.astype(np.int32), np.array([[0, 1, 2, 3]], dtype=np.int32), (n, n, n), (Ex,) * 3)
            assert_same(gpu_voxelize(m, tile=tile), cpu_voxelize(m), f"sweep k={k} d={d:.0f} tile={tile}")
            st = pkg.voxelize.last_status
            assert st["pairs"] >= 1
            flags.append(st["large_pairs"] / st["pairs"])
        assert all(f == 0.0 for f in flags[:10]), (tile, flags[:10])      # small end: int32 span records only
        assert all(f == 1.0 for f in flags[-10:]), (tile, flags[-10:])    # large end: int64 path only
        first_large = next(i for i, f in enumerate(flags) if f > 0)
        last_span = max(i for i, f in enumerate(flags) if f < 1)
        assert 10 <= first_large <= last_span + 1 <= 110, (tile, first_large, last_span)


def test_fast_setup_fit_test_is_straddled():
    """Round 2's fast plane setup is taken when 24*dx*dy*dz/g + 16*max(dy*dz*sx, dx*dz*sy, dx*dy*sz) < 2*10^9 (d = the tet's
    lattice bbox extents); everything else goes through the range-checked general setup.  Random tets whose
    extents sit around that bound, on power-of-two pitches (cubic and anisotropic), so that both routes -- and the
    general path's int32 / int64 split behind it -- meet in the same tiles.  The inequality is restated here only to
    assert that both sides occur; the expected grid is the oracle's."""
    fast = slow = 0
    for seed, (n, Ex) in enumerate([((128, 128, 128), (65536,) * 3), ((256, 256, 256), (16384,) * 3),
                                    ((128, 64, 32), (65536, 65536, 65536)), ((256, 256, 256), (1 << 20,) * 3)]):
        rng = np.random.default_rng(7000 + seed)
        h = [e // k for e, k in zip(Ex, n)]
        g = int(np.gcd.reduce(h))
        sx, sy, sz = (x // g for x in h)
        # extent at which a cubic bbox meets the bound: 24 d^3 / g + 16 d^2 s = 2e9
        d0 = int(min((2e9 * g / 24) ** (1 / 3), 30000))
        verts, tets = [], []
        for _ in range(400):
            size = int(d0 * 2 ** rng.uniform(-0.2, 1.4))
            c = np.array([rng.integers(0, e + 1) for e in Ex])
            pts = np.clip(c + rng.integers(-size // 2, size // 2 + 1, (4, 3)), 0, np.array(Ex))
            d = pts.max(0) - pts.min(0)
            if max(d) < 32768 and 24.0 * d[0] * d[1] * d[2] / g + 16.0 * max(d[1] * d[2] * sx, d[0] * d[2] * sy, d[0] * d[1] * sz) < 2.0e9:
                fast += 1
            else:
                slow += 1
            b = len(verts)
            verts += pts.tolist()
            tets.append([b, b + 1, b + 2, b + 3])
        m = Mesh(f"fit{seed}", np.array(verts, dtype=np.int32), np.array(tets, dtype=np.int32), n, Ex)
        exp = cpu_voxelize(m)
        assert_same(gpu_voxelize(m), exp, f"fit-test straddle {n} {Ex}")
        assert_same(gpu_voxelize(m, tile=(8, 8)), exp, f"fit-test straddle {n} {Ex} tile 8x8")
    assert fast > 400 and slow > 400, (fast, slow)


def test_more_meshes_than_griddim_z_holds():
    """K4 runs on a 3-D grid (tiles x, tiles y, tiles z * batch) when that fits gridDim and on a 1-D grid otherwise:
    66 000 meshes of 32 x 8 x 8 voxels (one tile each) take the 1-D launch.  Every third mesh holds a tet, the rest are
    empty."""
    B = 66000
    rng = np.random.default_rng(66)
    verts, tets, off = [], [], [0]
    for m_ in range(B):
        if m_ % 3 == 0:
            pts = rng.integers(0, [64 * 32 + 1, 64 * 8 + 1, 64 * 8 + 1], (4, 3))
            b = len(verts)
            verts += pts.tolist()
            tets.append([b, b + 1, b + 2, b + 3])
        off.append(len(tets))
    m = Mesh("manymeshes", np.array(verts, dtype=np.int32), np.array(tets, dtype=np.int32), (32, 8, 8), (64 * 32, 64 * 8, 64 * 8),
             tet_offsets=np.array(off, dtype=np.int64))
    assert m.batch == B
    exp = cpu_voxelize(m)
    assert exp.any()
    assert_same(gpu_voxelize(m), exp, "66000 meshes")


def test_more_oversized_tets_than_the_handover_list_holds():
    """Tets whose tile range exceeds 64 tiles are handed from K1 to K2's CTA through a 4096-entry list; with 5000 of
    them the rest falls back to the per-thread walk.  Both routes in one mesh, plus small tets."""
    import paper_2106_01326_b200 as pkg

    rng = np.random.default_rng(4096)
    verts, tets = [], []
    for i in range(5200):
        size = 36000 if i < 5000 else 900                  # ~70 voxels of 512 lattice units, or ~2 voxels
        c = rng.integers(0, E + 1, 3)
        pts = np.clip(c + rng.integers(-size // 2, size // 2 + 1, (4, 3)), 0, E)
        b = len(verts)
        verts += pts.tolist()
        tets.append([b, b + 1, b + 2, b + 3])
    m = Mesh("oversized", np.array(verts, dtype=np.int32), np.array(tets, dtype=np.int32), (128, 128, 128))
    exp = cpu_voxelize(m)
    assert_same(gpu_voxelize(m, tile=(8, 8)), exp, "oversized tile=(8,8)")
    assert pkg.voxelize.last_status["pairs"] > 64 * 4096
    assert_same(gpu_voxelize(m), exp, "oversized auto tile")
