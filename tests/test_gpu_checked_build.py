"""-m gpu: the CHECKED build of the library (libvox_checked.so, -DVOX_CHECKS) under the parity suite's small cases.

compute-sanitizer is closed on this pool (profiles/r02_sanitizers.md), so the kernels carry their own bounds checks:
every tile id, list entry, vertex id, record slot, image-row address, queue slot and grid word is tested before use
and the first violated check is reported by vox_debug_check_status.  Here a subprocess loads the checked library
(VOX_LIB) and runs the small-config, sparse, ragged, large-path, oversized-tet, randomized and lattice tests against
the oracle; it must finish green AND with no check violated.  A negative control shows that a violated check is seen."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SUBSET = ("small_configs or sparse_output or ragged or oversized or max_extent or straddle or randomized_jobs or "
          "unit_and_zero or random_soup or all_tets_culled or empty_mesh or p1_single or pipe_stream or "
          "gpu_lattice_input_matches or lattice_through_the_pipe or batched_lattice or fit_test or more_meshes or "
          "random_lattices or huge_index or graph_replay or swept_across or default_path_of_lattice or "
          "two_calls_in_a_row or built_in_workspace")


def _checked_lib():
    from paper_2106_01326_b200 import build

    return build.build_checked()


def test_parity_subset_under_the_checked_build():
    lib = _checked_lib()
    code = (
        "import json, sys, pytest\n"
        f"rc = pytest.main(['-q', '-x', '-m', 'gpu', '-p', 'no:cacheprovider', '-k', {SUBSET!r}, "
        "'tests/test_gpu_parity.py', 'tests/test_lattice.py', 'tests/test_zz_no_alloc.py'])\n"
        "import paper_2106_01326_b200 as pkg\n"
        "compiled, check = pkg.debug_check_status()\n"
        "print('CHECKED_RESULT ' + json.dumps({'rc': int(rc), 'compiled': compiled, 'check': check, 'lib': pkg.lib_path()}))\n"
    )
    env = dict(os.environ, VOX_LIB=lib)
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    lines = [l for l in out.stdout.splitlines() if l.startswith("CHECKED_RESULT ")]
    assert lines, out.stdout[-3000:] + out.stderr[-3000:]
    res = json.loads(lines[-1][len("CHECKED_RESULT "):])
    assert res["lib"] == lib and res["compiled"] is True, res
    assert res["rc"] == 0, out.stdout[-3000:]
    assert res["check"] == 0, f"device-side check {res['check']} was violated (codes: csrc/common.cuh CK_*)"


def test_a_violated_check_is_reported():
    """Negative control: tet indices beyond V (but inside the tensor, so the access itself is harmless)."""
    lib = _checked_lib()
    code = (
        "import json, numpy as np, torch\n"
        "import paper_2106_01326_b200 as pkg\n"
        "v = np.array([[0,0,0],[8192,0,0],[8192,8192,0],[8192,8192,8192]]*2, dtype=np.int32)\n"
        "t = np.array([[4,5,6,7]], dtype=np.int32)\n"
        "vz = pkg.Voxelizer((32,32,32))\n"
        "dv, dt = torch.from_numpy(v).cuda(), torch.from_numpy(t).cuda()\n"
        "vz._ck(vz._lib.vox_tets(vz._ctx, dv.data_ptr(), 4, dt.data_ptr(), 1, None), 'vox_tets')  # V = 4: ids 4..7 are out of range\n"
        "vz.run(); first = pkg.debug_check_status(); again = pkg.debug_check_status()\n"
        "print('CHECKED_RESULT ' + json.dumps({'first': first, 'again': again}))\n"
    )
    env = dict(os.environ, VOX_LIB=lib)
    out = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    lines = [l for l in out.stdout.splitlines() if l.startswith("CHECKED_RESULT ")]
    assert lines, out.stdout[-3000:] + out.stderr[-3000:]
    res = json.loads(lines[-1][len("CHECKED_RESULT "):])
    assert res["first"][0] is True and res["first"][1] in (102, 402), res   # a vertex-id check (K1 or K4)
    assert res["again"] == [True, 0], res                                   # reading clears it


def test_the_normal_build_compiles_no_checks():
    import paper_2106_01326_b200 as pkg

    if os.environ.get("VOX_LIB"):
        pytest.skip("running under VOX_LIB")
    assert pkg.debug_check_status() == (False, 0)
