"""-m gpu: full-size workloads of DESIGN.md "Input recipe" that tests/test_gpu_parity.py does not reach, element by element
against the oracle (SURVEY.md 8(d) "Caveat on cfgs 1, 5, S1, S2": a full box is all ones and cannot catch EXTRA bits, so every
full box also runs carved):

  * S2 = the Table-1-shaped meshes (10^5 / 10^6 / 10^7 tets at 256^3), full and with every third tet dropped;
  * S1 = 48 giant tets at its stated 512^3, full, every third tet dropped, and carved to a sphere;
  * cfg5 (graded stress: culled slivers + int64 pairs) carved two ways at 512^3, dense and sparse output;
  * lattice input (vox_lattice, vox_pipe_submit_lattice; dense and sparse) on the FULL cfg4 and cfg3, the workloads bench.py
    times it on.
"""
import functools

import numpy as np
import pytest

import meshgen
import oracle

pytestmark = pytest.mark.gpu
ONES = np.uint32(0xFFFFFFFF)


@functools.lru_cache(maxsize=3)
def _config(name):
    return meshgen.make_config(name)


@functools.lru_cache(maxsize=2)
def _expected(name):
    m = _config(name)
    return oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets)


def _cpu(m):
    return oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets)


def _gpu(m, **kw):
    import paper_2106_01326_b200 as pkg

    return pkg.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets if m.batch > 1 else None, **kw)


def assert_same(got, exp, what):
    if not np.array_equal(got, exp):
        bad = np.argwhere(got != exp)
        b = tuple(bad[0])
        raise AssertionError(
            f"{what}: {len(bad)} differing words; first at [m,z,y,xw]={b}: gpu={got[b]:#010x} oracle={exp[b]:#010x}; "
            f"popcount gpu={int(np.unpackbits(got.view(np.uint8)).sum())} "
            f"oracle={int(np.unpackbits(exp.view(np.uint8)).sum())}")


def _carve(m, how):
    if how == "full":
        return m
    if how == "drop3":
        return meshgen.carve_every_third(m)
    return meshgen.carve_sphere(m, 0.4 if how == "sphere" else 0.45)


# ------------------------------------------------------------------ S2: Table-1-shaped meshes at 256^3 (f2)
@pytest.mark.parametrize("how", ["full", "drop3"])
@pytest.mark.parametrize("name", ["s2_1e5", "s2_1e6", "s2_1e7"])
def test_table1_workloads_match_oracle(name, how):
    m = _carve(_config(name), how)
    exp = _cpu(m)
    got = _gpu(m)
    assert_same(got, exp, f"{name} {how}")
    if how == "full":
        assert np.all(got == ONES)               # P4: a conforming mesh of the closed box sets every bit
    else:
        assert not np.all(exp == ONES) and exp.any()


# ------------------------------------------------------------------ S1: giant tets at the stated 512^3
@pytest.mark.parametrize("how", ["full", "drop3", "sphere45"])
def test_giant_tets_at_512(how):
    m = _carve(_config("s1"), how)
    assert m.grid == (512, 512, 512)
    exp = _cpu(m)
    got = _gpu(m)
    assert_same(got, exp, f"s1 512^3 {how}")
    if how == "full":
        assert np.all(got == ONES)
    else:
        assert not np.all(exp == ONES) and exp.any()


# ------------------------------------------------------------------ cfg5 carved at full size, dense and sparse
@pytest.mark.parametrize("how", ["drop3", "sphere"])
def test_cfg5_carved_full_size_dense_and_sparse(how):
    import torch

    import paper_2106_01326_b200 as pkg
    from oracle import sparse

    m = _carve(_config("cfg5"), how)
    exp = _cpu(m)
    assert not np.all(exp == ONES) and exp.any()
    assert_same(_gpu(m), exp, f"cfg5 {how} dense")
    st = pkg.voxelize.last_status
    assert st["culled"] > 0 and st["large_pairs"] > 0      # the sliver cull and the int64 path are both exercised
    vz = pkg.Voxelizer(m.grid, m.extent, 1)
    try:
        vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda())
        vz.plan()
        ts = vz.tile_shape
        nb = ts["nbx"] * ts["nby"] * ts["nbz"]
        table, payload = vz.run_sparse(nb)
        sst = vz.sparse_status()
        table, payload = table.cpu().numpy().view(np.uint32), payload.cpu().numpy().view(np.uint32)
    finally:
        vz.close()
    assert sparse.check_table(table, payload, exp, ts["ty"], ts["tz"]) == sst["mixed_tiles"] > 0
    assert_same(sparse.decode(table, payload, m.grid, 1, ts["ty"], ts["tz"]), exp, f"cfg5 {how} sparse decode")


# ------------------------------------------------------------------ lattice input on the full bench workloads (f4)
def _pin(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


@pytest.mark.parametrize("variant", [0, 2], ids=["default", "fused"])
@pytest.mark.parametrize("name", ["cfg4", "cfg3"])
def test_lattice_input_full_size_device_and_pipe(name, variant):
    """vox_lattice (device pointers) and vox_pipe_submit_lattice (host buffers), dense and sparse, on the whole of
    cfg4 / cfg3 -- against the oracle on the tets written out, not against the tet-array GPU run.  The default takes
    the binning passes on these (cells of 8 and 2.7 voxels); variant 2 is the fused small-workspace path."""
    import torch

    import paper_2106_01326_b200 as pkg
    from oracle import sparse

    m = _config(name)
    exp = _expected(name)
    cells = m.cells
    keep = meshgen.lattice_form(m, cells)
    assert int(np.unpackbits(keep).sum()) == m.T
    d_verts, d_keep = torch.from_numpy(m.verts).cuda(), torch.from_numpy(keep).cuda()
    vz = pkg.Voxelizer(m.grid, m.extent, m.batch, variant=variant)
    try:
        vz.set_lattice(d_verts, cells, d_keep)
        assert vz.path == ("lattice_fused" if variant == 2 else "lattice_binned")
        vz.plan()
        got = vz.run().cpu().numpy().view(np.uint32)
        st = vz.status()
        assert_same(got, exp, f"{name} vox_lattice dense")
        ts = vz.tile_shape
        nb = m.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
        cap = max(int(st["nonempty_tiles"]), 1)
        table, payload = vz.run_sparse(cap)
        sst = vz.sparse_status()
        table, payload = table.cpu().numpy().view(np.uint32), payload.cpu().numpy().view(np.uint32)
        assert sparse.check_table(table, payload, exp, ts["ty"], ts["tz"]) == sst["mixed_tiles"] > 0
        assert_same(sparse.decode(table, payload, m.grid, m.batch, ts["ty"], ts["tz"]), exp, f"{name} vox_lattice sparse")
    finally:
        vz.close()
    del d_verts, d_keep
    lat_T = m.batch * 6 * cells[0] * cells[1] * cells[2]
    pipe = pkg.Pipe(m.grid, m.extent, m.batch, depth=2, max_V=m.V, max_T=lat_T, variant=variant)
    try:
        pts = pipe.tile_shape
        pnb = m.batch * pts["nbx"] * pts["nby"] * pts["nbz"]
        nx, ny, nz = m.grid
        h_out = torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32).pin_memory()
        h_tab = torch.zeros(pnb, dtype=torch.int32).pin_memory()
        h_pay = torch.zeros((pnb, pts["tz"], pts["ty"]), dtype=torch.int32).pin_memory()
        hv, hk = _pin(m.verts), _pin(keep)
        t0 = pipe.submit_lattice(hv, cells, hk, h_out)
        t1 = pipe.submit_lattice(hv, cells, hk, h_tab, h_pay, pnb)
        pipe.wait(t0)
        pst = pipe.wait(t1)
    finally:
        pipe.close()
    assert_same(h_out.numpy().view(np.uint32), exp, f"{name} pipe lattice dense")
    tb, pl = h_tab.numpy().view(np.uint32), h_pay.numpy().view(np.uint32)
    assert sparse.check_table(tb, pl, exp, pts["ty"], pts["tz"]) == pst["mixed_tiles"] > 0
    assert_same(sparse.decode(tb, pl, m.grid, m.batch, pts["ty"], pts["tz"]), exp, f"{name} pipe lattice sparse")
