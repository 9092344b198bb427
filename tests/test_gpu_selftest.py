"""-m gpu: the integer helpers of K4's row walk, operand by operand, against Python's exact integer division.

Whole-mesh parity finds a wrong helper late and by luck (a ptxas mis-fold corrupted this code twice).
The checked build (libvox_checked.so) exports vox_debug_selftest, which runs span_bound / recip_up / div_magic /
span64_bound -- the very device functions k4_flat inlines -- on operand arrays; expected values are plain `//`."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def checked():
    from paper_2106_01326_b200.build import build_checked

    lib = ctypes.CDLL(build_checked())
    lib.vox_debug_selftest.restype = ctypes.c_int
    lib.vox_debug_selftest.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                       ctypes.c_void_p]
    return lib


def run(lib, op, a, b):
    import torch

    a = np.ascontiguousarray(a, dtype=np.int64)
    b = np.ascontiguousarray(b, dtype=np.int64)
    assert a.shape == b.shape
    da, db = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    out = torch.full((a.size,), -12345, dtype=torch.int32, device="cuda")
    rc = lib.vox_debug_selftest(None, op, ctypes.c_void_p(da.data_ptr()), ctypes.c_void_p(db.data_ptr()), a.size,
                                ctypes.c_void_p(out.data_ptr()))
    assert rc == 1, rc
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.int64)


def divisors(rng):
    """a in {4..64} + {2^k - 1, 2^k, 2^k + 1} + random up to 2^31 - 1 (all >= 4)."""
    pw = np.array([(1 << k) + d for k in range(3, 31) for d in (-1, 0, 1)], dtype=np.int64)
    a = np.concatenate([np.arange(4, 65), pw, [(1 << 31) - 1, (1 << 31) - 2, (1 << 30) + 12345],
                        rng.integers(4, 1 << 31, 3000), rng.integers(4, 1 << 12, 1000)])
    return a[(a >= 4) & (a < (1 << 31))]


def operands(rng):
    """(r, a) pairs inside span_bound's contract: r at and around every kind of multiple of a, quotients up to 2^18 and
    beyond, negative r, and the largest |r| the set-up admits for that a (|r|(1 + 2^-18) + a < 2^31)."""
    rs, as_ = [], []
    for a in divisors(rng).tolist():
        rmax = int(((1 << 31) - 1 - a) / (1 + 2.0 ** -18)) - 1
        if rmax < 0:
            continue
        qmax = rmax // a
        qs = set([0, 1, 2, 3, 30, 31, 32, 33, 63, 64, 1000, (1 << 18) - 2, (1 << 18) - 1, 1 << 18, (1 << 18) + 1, qmax,
                  qmax - 1]) | set(rng.integers(0, max(qmax, 1) + 1, 24).tolist()) | set(rng.integers(0, 40, 8).tolist())
        for q in qs:
            if q < 0 or q > qmax:
                continue
            for d in (-2, -1, 0, 1, 2, a - 1, a // 2):
                r = q * a + d
                if -rmax <= r <= rmax:
                    rs.append(r)
                    as_.append(a)
        for r in (-1, -2, -a, -a - 1, -rmax, rmax, rmax - 1, -(rmax // 2)):
            rs.append(r)
            as_.append(a)
    return np.array(rs, dtype=np.int64), np.array(as_, dtype=np.int64)


@pytest.mark.parametrize("op", [0, 1], ids=["recip_up", "exact_reciprocal"])
def test_span_bound_against_integer_division(checked, op):
    rng = np.random.default_rng(5150 + op)
    r, a = operands(rng)
    assert len(r) > 100000
    got = run(checked, op, r, a)
    q = r // a                                  # numpy floor division on int64: exact
    small = (r >= 0) & (q < (1 << 18))
    assert small.sum() > 50000 and (~small).sum() > 10000
    bad = small & (got != q)
    assert not bad.any(), (int(bad.sum()), r[bad][:5], a[bad][:5], got[bad][:5], q[bad][:5])
    big = (r >= 0) & (q >= (1 << 18))
    assert (got[big] >= (1 << 18) - 1).all(), (r[big][got[big] < (1 << 18) - 1][:5], a[big][got[big] < (1 << 18) - 1][:5])
    neg = r < 0
    assert (got[neg] <= -1).all(), (r[neg][got[neg] > -1][:5], a[neg][got[neg] > -1][:5])


def test_recip_up_is_never_below_and_relatively_within_2_to_minus_19(checked):
    rng = np.random.default_rng(77)
    a = divisors(rng)
    inv = run(checked, 4, np.zeros_like(a), a)
    inv = inv & 0xFFFFFFFF                      # the helper returns the uint32 bit pattern in an int
    for ai, vi in zip(a.tolist(), inv.tolist()):   # Python integers: exact
        assert vi * ai >= (1 << 32), (ai, vi)                                         # never below 2^32 / a
        assert vi * ai * (1 << 19) < (1 << 32) * ((1 << 19) + 1) + ai * (1 << 19), (ai, vi)   # < (2^32/a)(1 + 2^-19) + 1
        assert vi < (1 << 31), (ai, vi)


def test_div_magic_exhaustively(checked):
    ny, rr = np.meshgrid(np.arange(1, 33), np.arange(0, 1024), indexing="ij")
    got = run(checked, 2, rr.ravel(), ny.ravel())
    assert np.array_equal(got, rr.ravel() // ny.ravel())


def test_span64_bound_against_integer_division(checked):
    rng = np.random.default_rng(64)
    a_list = np.concatenate([np.arange(1, 40), (1 << np.arange(1, 56)).astype(np.int64), (1 << np.arange(2, 56)).astype(np.int64) - 1,
                             rng.integers(1, 1 << 55, 4000), rng.integers(1, 1 << 20, 1000)]).astype(np.int64)
    q0s, as_ = [], []
    for a in a_list.tolist():
        for k in list(range(0, 35)) + [100, 1 << 10]:
            for d in (-1, 0, 1, a - 1, a // 2):
                q0 = k * a + d
                if q0 < (1 << 62):
                    q0s.append(q0)
                    as_.append(a)
        for q0 in (-1, -a, -(1 << 61)):
            q0s.append(q0)
            as_.append(a)
    q0, a = np.array(q0s, dtype=np.int64), np.array(as_, dtype=np.int64)
    got = run(checked, 3, q0, a)
    exp = np.where(q0 < 0, -1, np.minimum(q0 // a, 31))
    bad = got != exp
    assert not bad.any(), (int(bad.sum()), q0[bad][:5], a[bad][:5], got[bad][:5], exp[bad][:5])


def test_normal_build_compiles_no_selftest():
    import paper_2106_01326_b200 as pkg

    lib = pkg.load_library()
    if "checked" in pkg.lib_path():
        pytest.skip("running under the checked build")
    assert lib.vox_debug_selftest(None, 0, None, None, 0, None) == 0
