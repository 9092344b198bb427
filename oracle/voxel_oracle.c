/*
 * voxel_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU definition of the tetrahedral-mesh ->
 * solid-binary-voxel step of arxiv 2106.01326.  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may call
 * it.  It shares no code, header, table or helper with the CUDA path.
 *
 * What it computes:
 *
 *   bit(m,x,y,z) = OR over tets t of mesh m with 6V_t != 0 of inside(P, t)
 *   P = (hx*x + hx/2, hy*y + hy/2, hz*z + hz/2)            voxel centre (reading G7)
 *
 * following, in the paper's order and notation:
 *   - "voxelizing the tetrahedral mesh according to whether the sampling
 *     point is within a tetrahedral or not"
 *   - "We iterate over every bounding box of the tetrahedral and apply the
 *     ... point-in-tetrahedral test"
 *   - Theorem 1: a=PA, b=PB, c=PC, d=PD; D_a=det(b,c,d), D_b=det(a,c,d),
 *     D_c=det(a,b,d), D_d=det(a,b,c); inside <=> signs (+,-,+,-) or
 *     (-,+,-,+)
 *   - both orientation types (Lemma 1.1)
 *
 * Readings where the paper is silent:
 *   G1  the test is INCLUSIVE (>= / <=): closed tets, so a conforming mesh
 *       leaves no holes on shared faces;
 *   G2  degenerate tets (6V = det(B-A, C-A, D-A) == 0) contribute nothing;
 *   G8  closed bounding box, index range clamped to the grid;
 *   G9  x-fastest bit grid, 32 voxels per uint32, LSB = lowest x:
 *       word = ((m*nz + z)*ny + y)*(nx/32) + (x>>5), bit = x & 31.
 *
 * The determinants are evaluated DIRECTLY per sample by cofactor expansion in
 * int64_t: no incremental stepping, no bricks, no precomputed normals.
 * Coordinates in [0, 2^20] keep every intermediate below 2^63
 * (|det| <= 6 * (2^20)^3 < 2^63).
 *
 * mode 0: for tet: for voxel in clamped closed bbox
 * mode 1: for voxel: for tet (no bounding box at all)   (pins the bbox rounding)
 *
 * Parity pins: tests/test_oracle_pins.py (P1..P9), all independent of this file.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef int64_t i64;

static inline i64 det3(const i64 r0[3], const i64 r1[3], const i64 r2[3]) {
    return r0[0] * (r1[1] * r2[2] - r1[2] * r2[1])
         - r0[1] * (r1[0] * r2[2] - r1[2] * r2[0])
         + r0[2] * (r1[0] * r2[1] - r1[1] * r2[0]);
}

/* Theorem 1, inclusive (reading G1). */
static inline int inside_closed(const i64 P[3], const i64 A[3], const i64 B[3],
                                const i64 C[3], const i64 D[3]) {
    i64 a[3], b[3], c[3], d[3];
    for (int k = 0; k < 3; ++k) {
        a[k] = A[k] - P[k];
        b[k] = B[k] - P[k];
        c[k] = C[k] - P[k];
        d[k] = D[k] - P[k];
    }
    const i64 Da = det3(b, c, d);
    const i64 Db = det3(a, c, d);
    const i64 Dc = det3(a, b, d);
    const i64 Dd = det3(a, b, c);
    return (Da >= 0 && Db <= 0 && Dc >= 0 && Dd <= 0) ||
           (Da <= 0 && Db >= 0 && Dc <= 0 && Dd >= 0);
}

static inline i64 six_volume(const i64 A[3], const i64 B[3], const i64 C[3], const i64 D[3]) {
    i64 u[3], v[3], w[3];
    for (int k = 0; k < 3; ++k) {
        u[k] = B[k] - A[k];
        v[k] = C[k] - A[k];
        w[k] = D[k] - A[k];
    }
    return det3(u, v, w);
}

static inline i64 floor_div(i64 a, i64 b) { /* b > 0 */
    i64 q = a / b, r = a % b;
    return (r != 0 && r < 0) ? q - 1 : q;
}
static inline i64 ceil_div(i64 a, i64 b) { /* b > 0 */
    return -floor_div(-a, b);
}

static inline void load_tet(const int32_t* verts, const int32_t* tet, i64 A[3], i64 B[3],
                            i64 C[3], i64 D[3]) {
    for (int k = 0; k < 3; ++k) {
        A[k] = verts[3 * (i64)tet[0] + k];
        B[k] = verts[3 * (i64)tet[1] + k];
        C[k] = verts[3 * (i64)tet[2] + k];
        D[k] = verts[3 * (i64)tet[3] + k];
    }
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * verts [V][3], tets [T][4] (indices global into verts), tet_offsets [batch+1]
 * (mesh m owns tets tet_offsets[m] .. tet_offsets[m+1]-1).
 * bits: batch*nz*ny*(nx/32) words, fully overwritten.
 * tet_stride >= 1: only tets with (t % tet_stride) == 0 are processed (the
 *   bounded sample bench.py times; tests use 1).
 * samples_out (may be NULL): number of candidate samples visited = the
 *   paper's unit of work, sum over processed tets of |closed bbox ∩ centres|
 *   (mode 0) or voxels*tets (mode 1).
 * Returns 0, or -1 on invalid arguments.
 */
int oracle_voxelize(const int32_t* verts, i64 V, const int32_t* tets, i64 T,
                    const i64* tet_offsets, int batch, int nx, int ny, int nz, int ex, int ey,
                    int ez, int mode, i64 tet_stride, uint32_t* bits, i64* samples_out) {
    if (!bits || nx <= 0 || ny <= 0 || nz <= 0 || nx % 32 || batch < 1 || T < 0 || V < 0) return -1;
    if (ex % (2 * nx) || ey % (2 * ny) || ez % (2 * nz)) return -1;
    if (tet_stride < 1) return -1;
    const i64 h[3] = {ex / nx, ey / ny, ez / nz};
    const i64 n[3] = {nx, ny, nz};
    const i64 wpr = nx / 32;
    const i64 words_per_mesh = (i64)nz * ny * wpr;
    memset(bits, 0, sizeof(uint32_t) * (size_t)(words_per_mesh * batch));
    i64 samples = 0;

    for (int m = 0; m < batch; ++m) {
        const i64 t0 = tet_offsets ? tet_offsets[m] : 0;
        const i64 t1 = tet_offsets ? tet_offsets[m + 1] : T;
        uint32_t* grid = bits + words_per_mesh * m;
        if (mode == 0) {
#pragma omp parallel for schedule(dynamic, 256) reduction(+ : samples)
            for (i64 t = t0; t < t1; ++t) {
                if (t % tet_stride) continue;
                i64 A[3], B[3], C[3], D[3];
                load_tet(verts, tets + 4 * t, A, B, C, D);
                if (six_volume(A, B, C, D) == 0) continue; /* G2 */
                i64 i0[3], i1[3];
                int empty = 0;
                for (int k = 0; k < 3; ++k) {
                    i64 lo = A[k], hi = A[k];
                    if (B[k] < lo) lo = B[k];
                    if (C[k] < lo) lo = C[k];
                    if (D[k] < lo) lo = D[k];
                    if (B[k] > hi) hi = B[k];
                    if (C[k] > hi) hi = C[k];
                    if (D[k] > hi) hi = D[k];
                    /* centre c(i) = h*i + h/2 in [lo, hi]  (G8) */
                    i0[k] = ceil_div(2 * lo - h[k], 2 * h[k]);
                    i1[k] = floor_div(2 * hi - h[k], 2 * h[k]);
                    if (i0[k] < 0) i0[k] = 0;
                    if (i1[k] > n[k] - 1) i1[k] = n[k] - 1;
                    if (i0[k] > i1[k]) empty = 1;
                }
                if (empty) continue;
                samples += (i1[0] - i0[0] + 1) * (i1[1] - i0[1] + 1) * (i1[2] - i0[2] + 1);
                for (i64 z = i0[2]; z <= i1[2]; ++z)
                    for (i64 y = i0[1]; y <= i1[1]; ++y)
                        for (i64 x = i0[0]; x <= i1[0]; ++x) {
                            const i64 P[3] = {h[0] * x + h[0] / 2, h[1] * y + h[1] / 2,
                                              h[2] * z + h[2] / 2};
                            if (inside_closed(P, A, B, C, D)) {
                                uint32_t* w = grid + (z * ny + y) * wpr + (x >> 5);
                                __atomic_fetch_or(w, 1u << (x & 31), __ATOMIC_RELAXED);
                            }
                        }
            }
        } else {
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : samples)
            for (i64 z = 0; z < nz; ++z)
                for (i64 y = 0; y < ny; ++y)
                    for (i64 x = 0; x < nx; ++x) {
                        const i64 P[3] = {h[0] * x + h[0] / 2, h[1] * y + h[1] / 2,
                                          h[2] * z + h[2] / 2};
                        int hit = 0;
                        for (i64 t = t0; t < t1; ++t) {
                            if (t % tet_stride) continue;
                            i64 A[3], B[3], C[3], D[3];
                            load_tet(verts, tets + 4 * t, A, B, C, D);
                            ++samples;
                            if (six_volume(A, B, C, D) == 0) continue;
                            if (inside_closed(P, A, B, C, D)) hit = 1;
                        }
                        if (hit) grid[(z * ny + y) * wpr + (x >> 5)] |= 1u << (x & 31);
                    }
        }
    }
    if (samples_out) *samples_out = samples;
    return 0;
}

/* The four determinants and 6V for one (P, tet): exposed so the pins can test
 * the predicate identities (P5) against this exact code path. out[5] =
 * {Da, Db, Dc, Dd, 6V}. */
void oracle_determinants(const int32_t P_[3], const int32_t A_[3], const int32_t B_[3],
                         const int32_t C_[3], const int32_t D_[3], i64 out[5]) {
    i64 P[3], A[3], B[3], C[3], D[3], a[3], b[3], c[3], d[3];
    for (int k = 0; k < 3; ++k) {
        P[k] = P_[k]; A[k] = A_[k]; B[k] = B_[k]; C[k] = C_[k]; D[k] = D_[k];
        a[k] = A[k] - P[k]; b[k] = B[k] - P[k]; c[k] = C[k] - P[k]; d[k] = D[k] - P[k];
    }
    out[0] = det3(b, c, d);
    out[1] = det3(a, c, d);
    out[2] = det3(a, b, d);
    out[3] = det3(a, b, c);
    out[4] = six_volume(A, B, C, D);
}

int oracle_inside(const int32_t P_[3], const int32_t A_[3], const int32_t B_[3],
                  const int32_t C_[3], const int32_t D_[3]) {
    i64 P[3], A[3], B[3], C[3], D[3];
    for (int k = 0; k < 3; ++k) { P[k] = P_[k]; A[k] = A_[k]; B[k] = B_[k]; C[k] = C_[k]; D[k] = D_[k]; }
    if (six_volume(A, B, C, D) == 0) return 0;
    return inside_closed(P, A, B, C, D);
}
