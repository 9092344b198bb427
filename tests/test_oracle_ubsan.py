"""The oracle's int64 bound, checked by the compiler's own overflow trap (SURVEY.md section 5 "sanitizers").

oracle/voxel_oracle.c states that coordinates in [0, 2^20] keep every intermediate of Theorem 1's cofactor
determinants below 2^63 (|det| <= 6 * (2^20)^3 < 2^63).  Here the same source is built with
-fsanitize=signed-integer-overflow (trapping, not recovering) and driven at the largest extent the ABI admits with
tets that reach across the whole lattice, in both loop modes and through the single-point entry points; the
subprocess must exit 0.  liboracle.so itself is built WITHOUT -fwrapv, so an overflow would be undefined
behaviour there, not a silent wrap."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "voxel_oracle.c")

DRIVER = textwrap.dedent(
    r"""
    import ctypes, sys
    import numpy as np
    lib = ctypes.CDLL(sys.argv[1])
    i32p, i64p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int64)
    lib.oracle_voxelize.restype = ctypes.c_int
    lib.oracle_voxelize.argtypes = [i32p, ctypes.c_int64, i32p, ctypes.c_int64, i64p, ctypes.c_int] + [ctypes.c_int] * 7 + [
        ctypes.c_int64, ctypes.POINTER(ctypes.c_uint32), i64p]
    lib.oracle_determinants.restype = None
    lib.oracle_determinants.argtypes = [i32p] * 5 + [i64p]
    E = 1 << 20
    rng = np.random.default_rng(20)
    corners = np.array([[x, y, z] for x in (0, E) for y in (0, E) for z in (0, E)], dtype=np.int32)
    # every 4-subset of the lattice's corners (incl. the degenerate coplanar ones) + random giant and tiny tets
    import itertools
    tets = [list(c) for c in itertools.combinations(range(8), 4)]
    verts = [c for c in corners]
    for _ in range(200):
        size = int(rng.choice([E, E // 3, 4096, 37]))
        c = rng.integers(0, E + 1, 3)
        pts = np.clip(c + rng.integers(-size, size + 1, (4, 3)), 0, E)
        b = len(verts)
        verts += [p for p in pts]
        tets.append([b, b + 1, b + 2, b + 3])
    verts = np.ascontiguousarray(np.array(verts, dtype=np.int32))
    tets = np.ascontiguousarray(np.array(tets, dtype=np.int32))
    off = np.array([0, len(tets)], dtype=np.int64)
    total = 0
    for mode, n in ((0, 64), (1, 32)):
        bits = np.zeros((1, n, n, n // 32), dtype=np.uint32)
        samples = ctypes.c_int64(0)
        rc = lib.oracle_voxelize(verts.ctypes.data_as(i32p), len(verts), tets.ctypes.data_as(i32p), len(tets),
                                 off.ctypes.data_as(i64p), 1, n, n, n, E, E, E, mode, 1,
                                 bits.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)), ctypes.byref(samples))
        assert rc == 0
        assert np.all(bits == np.uint32(0xFFFFFFFF))       # the corner tets cover the whole box
        total += int(samples.value)
    # the extreme single-point cases: P on one corner, the tet on the others
    out = np.zeros(5, dtype=np.int64)
    for p in corners:
        for t in itertools.combinations(range(8), 4):
            a = [np.ascontiguousarray(corners[i]) for i in t]
            lib.oracle_determinants(np.ascontiguousarray(p).ctypes.data_as(i32p), *[x.ctypes.data_as(i32p) for x in a],
                                    out.ctypes.data_as(i64p))
            assert abs(int(out[4])) <= 6 * E ** 3
    print("ok", total)
    """
)


def test_oracle_has_no_signed_overflow_at_the_largest_extent(tmp_path):
    lib = str(tmp_path / "liboracle_ubsan.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-fopenmp", "-fsanitize=signed-integer-overflow",
                           "-fsanitize-undefined-trap-on-error", "-shared", "-fPIC", "-o", lib, SRC])
    drv = tmp_path / "drive.py"
    drv.write_text(DRIVER)
    r = subprocess.run([sys.executable, str(drv), lib], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, f"overflow trap or failure (rc {r.returncode}):\n{r.stdout}\n{r.stderr}"
    assert r.stdout.startswith("ok")


def test_overflow_trap_fires_when_the_bound_is_exceeded(tmp_path):
    """The trap is live: the same build aborts when driven beyond the documented bound (coordinates of 2^30)."""
    lib = str(tmp_path / "liboracle_ubsan.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-fopenmp", "-fsanitize=signed-integer-overflow",
                           "-fsanitize-undefined-trap-on-error", "-shared", "-fPIC", "-o", lib, SRC])
    code = textwrap.dedent(
        r"""
        import ctypes, sys
        import numpy as np
        lib = ctypes.CDLL(sys.argv[1])
        i32p, i64p = ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int64)
        lib.oracle_determinants.restype = None
        lib.oracle_determinants.argtypes = [i32p] * 5 + [i64p]
        B = 1 << 30
        pts = [np.array(v, dtype=np.int32) for v in ((0, 0, 0), (B, 0, 0), (0, B, 0), (0, 0, B), (B, B, B))]
        out = np.zeros(5, dtype=np.int64)
        lib.oracle_determinants(*[p.ctypes.data_as(i32p) for p in (pts[4], pts[0], pts[1], pts[2], pts[3])],
                                out.ctypes.data_as(i64p))
        print("survived")
        """
    )
    drv = tmp_path / "beyond.py"
    drv.write_text(code)
    r = subprocess.run([sys.executable, str(drv), lib], capture_output=True, text=True, timeout=120)
    assert r.returncode != 0 and "survived" not in r.stdout
