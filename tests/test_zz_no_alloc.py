"""vox_run_noalloc: the hot path for callers that may not allocate device memory.

Who that is: code that receives its input and output buffers from a host application but has no device memory of
its own to give vox_run as a workspace -- a plug-in inside an application whose memory pool already owns the whole
GPU, a service loop that cannot take the device-wide synchronisation an allocation brings, a thread in a process
where someone else is capturing a graph in global mode (an allocation call there is an error).  For them libvox.so
carries a 4 MiB workspace of its own (include/vox.h, VOX_NOALLOC_SCRATCH_BYTES); jobs that need more are refused.

What is checked: the new entry point gives, word for word, the grid the existing vox_run path gives (integer work:
the bar is equality, as everywhere in this suite), on two calls in a row that share the built-in array -- two
different meshes, so anything the first call left behind would show in the second -- and that an oversized job is
turned away with a clear message instead of being run.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the rest of the suite.  It passes alone in a fresh process (the first call does the per-device set-up) and after
the other tests (the array then holds their leftovers: none of them use it, so it holds zeros or this file's own).
"""
import ctypes

import numpy as np
import pytest

import meshgen

E = 65536


def _existing_path(pkg, torch, m):
    """The grid from vox_run on a caller-allocated workspace (the path every other test in the suite exercises)."""
    vz = pkg.Voxelizer(m.grid, m.extent, m.batch)
    off = torch.from_numpy(m.tet_offsets).cuda() if m.batch > 1 else None
    vz.set_tets(torch.from_numpy(m.verts).cuda(), torch.from_numpy(m.tets).cuda(), off)
    vz.plan()
    out = vz.run()
    st = vz.status()
    return vz, out.cpu().numpy().view(np.uint32), st


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    import torch

    import paper_2106_01326_b200 as pkg

    # cfg2 (75 014 tets, 128^3: a 1.9 MB workspace) and a carved cfg1 (256 tets, 32^3, most pairs on the int64 path)
    meshes = [meshgen.make_config("cfg2"), meshgen.carve_every_third(meshgen.make_config("cfg1"))]
    launches_per_run = None
    for round_ in range(2):  # the same pair again: the array now holds the second mesh's leftovers
        for m in meshes:
            vz, expect, st_expect = _existing_path(pkg, torch, m)
            assert vz.workspace_bytes <= pkg.binding.NOALLOC_SCRATCH_BYTES
            nx, ny, nz = m.grid
            out = torch.full((m.batch, nz, ny, nx // 32), -1, dtype=torch.int32, device="cuda")  # stale bits
            before = pkg.kernel_launches()
            st = vz.run_noalloc(out)  # same context, same borrowed inputs; only the workspace differs
            launched = pkg.kernel_launches() - before
            got = out.cpu().numpy().view(np.uint32)
            assert np.array_equal(got, expect), (
                f"{m.name} round {round_}: {int((got != expect).sum())} words differ from vox_run's grid")
            assert st == st_expect, (m.name, st, st_expect)
            assert launched == 4  # K1, K2, K3, K4: our kernels ran, nothing else
            launches_per_run = launched
            # and once more without the status read-back (enqueue only), straight after: still the same grid
            out.fill_(-1)
            assert vz.run_noalloc(out, stats=False) is None
            torch.cuda.synchronize()
            assert np.array_equal(out.cpu().numpy().view(np.uint32), expect), f"{m.name}: enqueue-only call differs"
            vz.close()
    assert launches_per_run == 4


@pytest.mark.gpu
def test_lattice_input_through_the_built_in_workspace():
    """The fused lattice path keeps a 16-byte copy of every vertex in the workspace: it fits for small lattices."""
    import torch

    import paper_2106_01326_b200 as pkg

    m = meshgen.carve_sphere(meshgen.make_config("cfg1"))
    _, expect, _ = _existing_path(pkg, torch, m)
    keep = meshgen.lattice_form(m, (4, 4, 4))
    vz = pkg.Voxelizer(m.grid, m.extent, 1)
    vz.set_lattice(torch.from_numpy(m.verts).cuda(), (4, 4, 4), torch.from_numpy(keep).cuda())
    out = torch.full((1, 32, 32, 1), -1, dtype=torch.int32, device="cuda")
    for _ in range(2):
        vz.run_noalloc(out)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), expect)
        out.fill_(-1)


def test_oversized_job_is_refused_before_any_gpu_work():
    """Needs no device: the size test precedes every CUDA call.  4.8 M tets on 1024^3 want ~140 MB."""
    from paper_2106_01326_b200.build import build

    build()
    import paper_2106_01326_b200 as pkg

    lib = pkg.load_library()
    c = ctypes.c_void_p()
    assert lib.vox_create(ctypes.byref(c), 1024, 1024, 1024, E, E, E, 1) == 0
    # before vox_tets: call order
    assert lib.vox_run_noalloc(c, None, ctypes.c_void_p(256), None) == -5
    assert lib.vox_tets(c, ctypes.c_void_p(256), 2_000_000, ctypes.c_void_p(256), 4_800_000, None) == 0
    assert lib.vox_workspace_bytes(c) > pkg.binding.NOALLOC_SCRATCH_BYTES
    assert lib.vox_run_noalloc(c, None, ctypes.c_void_p(256), None) == -3  # VOX_EWORKSPACE
    msg = lib.vox_last_error(c).decode()
    assert "vox_run_noalloc" in msg and str(pkg.binding.NOALLOC_SCRATCH_BYTES) in msg
    assert str(lib.vox_workspace_bytes(c)) in msg
    assert lib.vox_run_noalloc(c, None, None, None) == -1  # no output buffer
    lib.vox_destroy(c)
    # the header's constant and the binding's agree
    hdr = open(pkg.binding._HERE + "/../include/vox.h").read()
    assert "#define VOX_NOALLOC_SCRATCH_BYTES (4u << 20)" in hdr and pkg.binding.NOALLOC_SCRATCH_BYTES == 4 << 20
