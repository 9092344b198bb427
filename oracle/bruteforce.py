"""Second, independent oracle: pure-Python big integers, no bounding box.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  For tiny inputs only (every voxel centre
is tested against every tet).  It restates the definition of DESIGN.md "Oracle"
without sharing a line with ``voxel_oracle.c``: the determinants are written as
scalar triple products a . (b x c) instead of a cofactor expansion, and there is
no bounding box, no clamping and no fixed-width integer anywhere.

  Theorem 1: a=PA, b=PB, c=PC, d=PD,
  D_a=det(b,c,d), D_b=det(a,c,d), D_c=det(a,b,d), D_d=det(a,b,c);
  inside <=> signs (+,-,+,-) or (-,+,-,+); made inclusive (reading G1);
  tets with 6V = det(AB,AC,AD) = 0 contribute nothing (reading G2).
"""
from __future__ import annotations

import numpy as np


def _sub(u, v):
    return (u[0] - v[0], u[1] - v[1], u[2] - v[2])


def _cross(u, v):
    return (u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0])


def _dot(u, v):
    return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]


def _triple(u, v, w):
    """det of the matrix with rows u, v, w = u . (v x w)."""
    return _dot(u, _cross(v, w))


def inside_closed_py(P, A, B, C, D) -> bool:
    P, A, B, C, D = (tuple(int(x) for x in q) for q in (P, A, B, C, D))
    if _triple(_sub(B, A), _sub(C, A), _sub(D, A)) == 0:
        return False
    a, b, c, d = _sub(A, P), _sub(B, P), _sub(C, P), _sub(D, P)
    Da, Db, Dc, Dd = _triple(b, c, d), _triple(a, c, d), _triple(a, b, d), _triple(a, b, c)
    return (Da >= 0 and Db <= 0 and Dc >= 0 and Dd <= 0) or (
        Da <= 0 and Db >= 0 and Dc <= 0 and Dd >= 0
    )


def bruteforce_voxelize(verts, tets, grid, extent=(65536, 65536, 65536), strict=False):
    """uint32[nz][ny][nx/32] for ONE mesh; all voxels x all tets.

    strict=True applies Theorem 1 literally (open tet) -- used only by the pin
    that shows why the inclusive reading G1 is needed.
    """
    nx, ny, nz = grid
    ex, ey, ez = extent
    assert ex % (2 * nx) == 0 and ey % (2 * ny) == 0 and ez % (2 * nz) == 0 and nx % 32 == 0
    hx, hy, hz = ex // nx, ey // ny, ez // nz
    V = [tuple(int(c) for c in v) for v in np.asarray(verts).reshape(-1, 3)]
    T = [tuple(int(i) for i in t) for t in np.asarray(tets).reshape(-1, 4)]
    live = []
    for t in T:
        A, B, C, D = (V[i] for i in t)
        if _triple(_sub(B, A), _sub(C, A), _sub(D, A)) != 0:
            live.append((A, B, C, D))
    bits = np.zeros((nz, ny, nx // 32), dtype=np.uint32)
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                P = (hx * x + hx // 2, hy * y + hy // 2, hz * z + hz // 2)
                hit = False
                for A, B, C, D in live:
                    a, b, c, d = _sub(A, P), _sub(B, P), _sub(C, P), _sub(D, P)
                    Da = _triple(b, c, d)
                    Db = _triple(a, c, d)
                    Dc = _triple(a, b, d)
                    Dd = _triple(a, b, c)
                    if strict:
                        ok = (Da > 0 and Db < 0 and Dc > 0 and Dd < 0) or (
                            Da < 0 and Db > 0 and Dc < 0 and Dd > 0)
                    else:
                        ok = (Da >= 0 and Db <= 0 and Dc >= 0 and Dd <= 0) or (
                            Da <= 0 and Db >= 0 and Dc <= 0 and Dd >= 0)
                    if ok:
                        hit = True
                        break
                if hit:
                    bits[z, y, x >> 5] |= np.uint32(1 << (x & 31))
    return bits
