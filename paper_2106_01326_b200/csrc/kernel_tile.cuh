// kernel_tile.cuh -- part of vox.cu (included there, once): K4/K5 building blocks: planes, pair records, set-up paths, span arithmetic, row walk, tile epilogue.
#pragma once

// ------------------------------------------------------------------------------------------
// K4: tile voxelizer
// ------------------------------------------------------------------------------------------
// The four half-spaces of a non-degenerate tet, written on tile-local voxel indices j:
//   inside(j) <=> G_k(j) = g0[k] + mx[k]*jx + my[k]*jy + mz[k]*jz >= 0,  k = 0..3.
// Derivation: Theorem 1's determinants are affine in P:
//   D_a = N_a.(B-P), N_a=(C-B)x(D-B);  D_b = N_b.(A-P), N_b=(C-A)x(D-A);
//   D_c = N_c.(A-P), N_c=(B-A)x(D-A);  D_d = N_d.(A-P), N_d=(B-A)x(C-A);
// with s = sign(6V): inside <=> s*D_a >= 0, -s*D_b >= 0, s*D_c >= 0, -s*D_d >= 0.
// P = h*(i0+j) + h/2 (componentwise), g = gcd(h): sigma*N.(Q-P) = C - g * sum_a (sigma*N_a*h_a/g) j_a
// with C = sigma*N.(Q-P0) and the j-sum an integer, so  >= 0  <=>  floor(C/g) - sum >= 0.
struct Planes {
    i64 mx[4], my[4], mz[4], g0[4];
};

__device__ __forceinline__ void one_plane(const Params& p, int k, Planes& P, i64 sig, i64 px, i64 py, i64 pz,
                                          i64 qx, i64 qy, i64 qz,  // N = p x q
                                          i64 rx, i64 ry, i64 rz)  // Q - P0
{
    i64 nx = sig * (py * qz - pz * qy);
    i64 ny = sig * (pz * qx - px * qz);
    i64 nz = sig * (px * qy - py * qx);
    i64 C = nx * rx + ny * ry + nz * rz;
    P.mx[k] = -nx * p.sx;
    P.my[k] = -ny * p.sy;
    P.mz[k] = -nz * p.sz;
    P.g0[k] = (p.g_shift >= 0) ? (C >> p.g_shift) : floor_div_l(C, (i64)p.g);
}

// X0,Y0,Z0: voxel index of the tile origin
__device__ __forceinline__ void tet_planes(const Params& p, const Tet& q, int X0, int Y0, int Z0, Planes& P) {
    i64 ux = q.bx - q.ax, uy = q.by - q.ay, uz = q.bz - q.az;
    i64 vx = q.cx - q.ax, vy = q.cy - q.ay, vz = q.cz - q.az;
    i64 wx = q.dx - q.ax, wy = q.dy - q.ay, wz = q.dz - q.az;
    i64 det = ux * (vy * wz - vz * wy) - uy * (vx * wz - vz * wx) + uz * (vx * wy - vy * wx);
    i64 s = (det > 0) ? 1 : -1;
    // P0 = centre of the tile-origin voxel
    i64 p0x = (i64)p.hx * X0 + (p.hx >> 1), p0y = (i64)p.hy * Y0 + (p.hy >> 1), p0z = (i64)p.hz * Z0 + (p.hz >> 1);
    i64 arx = q.ax - p0x, ary = q.ay - p0y, arz = q.az - p0z;
    i64 brx = q.bx - p0x, bry = q.by - p0y, brz = q.bz - p0z;
    // k=0: s * ((C-B)x(D-B)) . (B-P)
    one_plane(p, 0, P, s, vx - ux, vy - uy, vz - uz, wx - ux, wy - uy, wz - uz, brx, bry, brz);
    // k=1: -s * ((C-A)x(D-A)) . (A-P)
    one_plane(p, 1, P, -s, vx, vy, vz, wx, wy, wz, arx, ary, arz);
    // k=2: s * ((B-A)x(D-A)) . (A-P)
    one_plane(p, 2, P, s, ux, uy, uz, wx, wy, wz, arx, ary, arz);
    // k=3: -s * ((B-A)x(C-A)) . (A-P)
    one_plane(p, 3, P, -s, ux, uy, uz, vx, vy, vz, arx, ary, arz);
}

__device__ __forceinline__ i64 iabs64(i64 v) { return v < 0 ? -v : v; }


// ------------------------------------------------------------------------------------------
// K4: row-span voxelizer.  DESIGN.md "Kernels / K4".
// Inside a tile row (y,z) every half-space G_k(x) = r_k + mx_k*x >= 0 is a half-line in x, so the
// row's solid set is ONE interval [lower, upper].  Each plane is stored as a function Q that is
// non-increasing in x and whose non-negative set {x : Q(x) >= 0} is
//   hi-type (mx_G < 0): Q = G                     -> x <= b,  b = max{x : G(x) >= 0}
//   lo-type (mx_G > 0): Q = -G - 1  (G <= -1)     -> x <= b  <=> G(x) < 0, so the half-space is x >= b+1
//   mx_G == 0:          r' = 64*G + 63, mx = 0 (hi) -> gates the row only (see span_plane)
// b = floor of the real crossing r/|mx|.  A fixed-point reciprocal PROPOSES c0 = floor(r*inv/2^32) >= B, which
// is B or B+1 whenever B < 2^18 (see span_bound); the INTEGER value Q(c0) decides: b = c0 if Q(c0) >= 0 else c0-1.
// Planes are stored scaled by 4 so that |mx| >= 4 and the reciprocal fits int32; every row value r of the
// pair's box and r +- 2*mx fit int32 (guaranteed at setup, see setup_pair / span_plane).
// ------------------------------------------------------------------------------------------
// Record of one (tet, tile) pair in shared memory, 40 words:
//   [0..3]   A = x0+1, x1-x0, ny, nrows          (box-relative: rows (yy,zz) and x' = x - x0 count from the pair's box)
//   [4..7]   B = shared byte address of image row (y0,z0), div-by-ny magic, c1, c2
//            (c1 / c2: plane slot 1 / 2 is lo-type ? +2^30 : -2^30;  c1 == 0 marks a LARGE record, B.y = its box)
//   [8..23]  four plane slots {mx, my, mz, g0 (at the box origin)}, lo-types first: slot 0 is always lo, slot 3 always hi
//   [24..27] ceil-ish 2^32/|mx| of the four slots
//   large records: [8..39] the 16 int64 values mx[4], my[4], mz[4], g0[4] of tet_planes (tile-relative)
// Record pi starts at word pi*40 + 4*(pi/4): the 16-byte pad after every fourth record puts the same 16-byte
// chunk of eight consecutive records into eight different bank groups (2*pi + pi/4 mod 8 is a bijection on
// 0..7), so the LDS.128 / STS.128 of lanes that sit in neighbouring records do not conflict (stride 40 alone
// gave two-way conflicts: profiles/r02a).
// image: row (y,z) of the tile lives at img[z*(TY+IMG_SKEW) + y] (skew spreads a tet's rows over banks)
enum { SREC_W = 40, IMG_SKEW = 11 };
#define REC_WORDS(NT) ((NT) * SREC_W + ((NT) / 4) * 4)
__device__ __forceinline__ int rec_off(int pi) { return pi * SREC_W + ((pi >> 2) << 2); }
#define LARGE_W(i) (8 + 2 * (i))

// per-CTA constants of the tile
struct TileGeo {
    int X0, Y0, Z0;       // voxel index of the tile origin
    int ymax, zmax;       // last row / slice of the tile that lies inside the grid (tile-local)
    int p0x, p0y, p0z;    // lattice coordinates of the centre of the tile-origin voxel
    int img_stride;
    u32 img_saddr;
};

__device__ __forceinline__ u32 pack_box(int x0, int x1, int y0, int y1, int z0, int z1) {
    return (u32)x0 | ((u32)x1 << 5) | ((u32)y0 << 10) | ((u32)y1 << 15) | ((u32)z0 << 20) | ((u32)z1 << 25);
}

// a record that draws nothing: one row whose upper bound is -2 (plane slots are never looked at: n < 0 whatever they hold)
__device__ __forceinline__ void null_record(int* rec, u32 img_saddr) {
    *reinterpret_cast<int4*>(rec) = make_int4(1, -2, 1, 1);
    *reinterpret_cast<int4*>(rec + 4) = make_int4((int)img_saddr, 0, 1 << 30, -(1 << 30));
}

// One plane of the span record, general path.  (nx,ny,nz) = sigma*N (int32, exact), (rx,ry,rz) = Q - P0 (P0 = centre
// of the tile-origin voxel).  G(j) = floor(C/g) - sum_a (sigma*N_a*s_a) j_a, C = sigma*N.(Q-P0)
// The record is written relative to the pair's local box: row (yy,zz), x' = x - x0, so that the stored
// values are distances from the BOX (not the tile) origin and small tets stay in int32 on coarse lattices.
__device__ __forceinline__ bool span_plane(const Params& p, int* rec, int pos, int nx, int ny, int nz, int rx, int ry,
                                           int rz, int x0, int y0, int z0, int wy, int wz) {
    // 64-bit only where the VALUE needs it (C and the box-origin shift); everything else is 32-bit once the
    // coefficients are known to fit.  Anything that does not fit returns false -> exact int64 large path.
    bool ok = (abs(nx) <= p.lim_x) && (abs(ny) <= p.lim_y) && (abs(nz) <= p.lim_z);  // |m| < 2^30
    // (unsigned products: no signed overflow when a component is out of range and ok is already false)
    int mx = (int)(0u - (u32)nx * (u32)p.sx), my = (int)(0u - (u32)ny * (u32)p.sy), mz = (int)(0u - (u32)nz * (u32)p.sz);
    const i64 C = (i64)nx * rx + (i64)ny * ry + (i64)nz * rz;
    const i64 g64 = (C >> p.g_shift) + (i64)mx * x0 + (i64)my * y0 + (i64)mz * z0;  // G at the box origin
    ok = ok && ((u64)(g64 + (1ll << 31) - 1) < (1ull << 32) - 2);                  // |g0| < 2^31 (acc below bounds it further)
    int g0 = (int)g64;
    if (mx > 0) { mx = (int)(0u - (u32)mx); my = (int)(0u - (u32)my); mz = (int)(0u - (u32)mz); g0 = ~g0; }  // lo-type: Q = -G - 1
    // scale: 4 (when |mx| < 4), so that |mx| >= 4 and the reciprocal ceil(2^32 / |mx|) fits int32; a plane with mx == 0 does
    // not depend on x and only gates the row: stored as r' = 64*G + 63 with inv = 2^31 - 1, for which span_bound
    // gives c0 = floor(r'/2 - r'/2^32) >= 31 when r' >= 63 (G >= 0: not binding, x1' <= 31) and b = c0 - 1 <= -2
    // when r' <= -1 (G < 0: empty row).
    // (every x-dependent plane is scaled by 4, not "2, or 4 when |mx| == 1": ptxas 12.9 at -O1 and above folds the
    //  test `mx == -1` on the negated absolute value to false -- SASS keeps only the cases 1 and 6 -- which the
    //  parity suite caught twice)
    // (general path, round 2: a plane whose |mx| is already >= 4 is not scaled at all -- two more bits of headroom before
    //  a pair has to take the int64 path: the Table-1 mesh of 10^5 tets had 41 043 such pairs)
    const int sh = (mx == 0) ? 6 : (((u32)0 - (u32)mx) >= 4u ? 0 : 2);
    // every row value r of the box and r +- 2*mx (span_bound's product and check) must fit int32 after scaling
    u64 acc = (u64)(u32)abs(g0) + 2ull * (0u - (u32)mx);
    acc += (u64)(u32)wy * (u32)abs(my);
    acc += (u64)(u32)wz * (u32)abs(mz);
    ok = ok && (acc < (u64)((0x7FFFFF00u - 63u) >> sh));
    mx = (int)((u32)mx << sh);
    my = (int)((u32)my << sh);
    mz = (int)((u32)mz << sh);
    g0 = (int)((u32)g0 << sh) + ((sh == 6) ? 63 : 0);
    const u32 a = max((u32)(-mx), 4u);  // a valid plane with mx != 0 has |mx| >= 4 after scaling
    const u32 inv = (sh == 6) ? 0x7FFFFFFFu : (0xFFFFFFFFu / a) + 1u;  // in [2^32/a, 2^32/a + 1), < 2^31
    *reinterpret_cast<int4*>(rec + 8 + 4 * pos) = make_int4(mx, my, mz, g0);
    rec[24 + pos] = (int)inv;
    return ok;
}

// record of a large pair: header A = one row that draws nothing (x1' = -2), so that the row walk of k4_flat steps
// over the pair like over any other; B = image address, packed local box, 0 (= large), 0; words 8..39 the int64 planes
__device__ __noinline__ void large_record(const Params& p, const Tet& q, const TileGeo& g, u32 box, int* rec) {
    Planes P;
    tet_planes(p, q, g.X0, g.Y0, g.Z0, P);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        *reinterpret_cast<i64*>(rec + LARGE_W(k)) = P.mx[k];
        *reinterpret_cast<i64*>(rec + LARGE_W(4 + k)) = P.my[k];
        *reinterpret_cast<i64*>(rec + LARGE_W(8 + k)) = P.mz[k];
        *reinterpret_cast<i64*>(rec + LARGE_W(12 + k)) = P.g0[k];
    }
    *reinterpret_cast<int4*>(rec) = make_int4(0, -2, 1, 1);
    *reinterpret_cast<int4*>(rec + 4) = make_int4((int)g.img_saddr, (int)box, 0, 0);
}

// b = max{x in [0,31] : q0 - a*x >= 0}, or -1 if there is none (a > 0).  A float quotient PROPOSES (its error is
// far below 1 for quotients up to 32), the exact int64 value decides; quotients beyond 31 saturate.
__device__ __forceinline__ int span64_bound(i64 q0, i64 a) {
    if (q0 < 0) return -1;
    int c = (int)fminf(__ll2float_rn(q0) / __ll2float_rn(a), 31.0f);
    const i64 v = q0 - a * c;
    if (v < 0) c -= 1;
    else if (c < 31 && v - a >= 0) c += 1;
    return c;
}

// rasterise one large pair from the int64 planes in its record (large_record): one warp
__device__ __noinline__ void raster_large_rec(const int* rec, u32* img, int lane, int img_stride) {
    Planes P;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        P.mx[k] = *reinterpret_cast<const i64*>(rec + LARGE_W(k));
        P.my[k] = *reinterpret_cast<const i64*>(rec + LARGE_W(4 + k));
        P.mz[k] = *reinterpret_cast<const i64*>(rec + LARGE_W(8 + k));
        P.g0[k] = *reinterpret_cast<const i64*>(rec + LARGE_W(12 + k));
    }
    const u32 box = (u32)rec[5];
    const int x0 = box & 31, x1 = (box >> 5) & 31, y0 = (box >> 10) & 31, y1 = (box >> 15) & 31;
    const int z0 = (box >> 20) & 31, z1 = (box >> 25) & 31;
    VOX_CHECK(x0 <= x1 && y0 <= y1 && z0 <= z1 && (z1 * img_stride + y1) < 32 * (32 + IMG_SKEW), CK_K4_LARGEBOX);
    bool all_in = true, any_out = false;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        i64 ax0 = P.mx[k] * x0, ax1 = P.mx[k] * x1, ay0 = P.my[k] * y0, ay1 = P.my[k] * y1;
        i64 az0 = P.mz[k] * z0, az1 = P.mz[k] * z1;
        i64 lo = P.g0[k] + min(ax0, ax1) + min(ay0, ay1) + min(az0, az1);
        i64 hi = P.g0[k] + max(ax0, ax1) + max(ay0, ay1) + max(az0, az1);
        all_in = all_in && (lo >= 0);
        any_out = any_out || (hi < 0);
    }
    if (any_out) return;  // one half-space misses the whole box: exact, G is affine
    const u32 xmask = (0xFFFFFFFFu >> (31 - x1 + x0)) << x0;
    const int ny = y1 - y0 + 1;
    if (all_in) {  // the box lies inside the tet
        const int nrows = ny * (z1 - z0 + 1);
        for (int r = lane; r < nrows; r += 32) {
            int zz = r / ny;
            atomicOr(img + (z0 + zz) * img_stride + y0 + r - zz * ny, xmask);
        }
        return;
    }
    const int nrows = ny * (z1 - z0 + 1);
    if (nrows > 5) {
        // many rows: lanes = rows, each lane finds its row's span from four exact int64 bounds (span64_bound)
        for (int r = lane; r < nrows; r += 32) {
            const int zz = r / ny;
            const int y = y0 + r - zz * ny, z = z0 + zz;
            int lower = x0 - 1, upper = x1;  // solid x in (lower, upper]
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const i64 G0 = P.g0[k] + P.my[k] * y + P.mz[k] * z;  // G at x = 0 of this row
                if (P.mx[k] > 0) lower = max(lower, span64_bound(-G0 - 1, P.mx[k]));          // G(x) >= 0 <=> x >= b + 1
                else if (P.mx[k] < 0) upper = min(upper, span64_bound(G0, -P.mx[k]));         // G(x) >= 0 <=> x <= b
                else if (G0 < 0) upper = -2;                                                   // x-independent plane
            }
            const int n = upper - lower;
            if (n > 0) atomicOr(img + z * img_stride + y, (0xFFFFFFFFu >> (32 - n)) << (lower + 1));
        }
        return;
    }
    // few rows: lanes = the 32 x positions of a row word, __ballot_sync forms the word
    i64 c0 = P.g0[0] + P.mx[0] * lane, c1 = P.g0[1] + P.mx[1] * lane;
    i64 c2 = P.g0[2] + P.mx[2] * lane, c3 = P.g0[3] + P.mx[3] * lane;
    for (int z = z0; z <= z1; ++z) {
        i64 r0 = c0 + P.mz[0] * z + P.my[0] * y0, r1 = c1 + P.mz[1] * z + P.my[1] * y0;
        i64 r2 = c2 + P.mz[2] * z + P.my[2] * y0, r3 = c3 + P.mz[3] * z + P.my[3] * y0;
        for (int y = y0; y <= y1; ++y) {
            u32 word = __ballot_sync(0xFFFFFFFFu, (r0 | r1 | r2 | r3) >= 0) & xmask;
            if (lane == 0 && word) atomicOr(img + z * img_stride + y, word);
            r0 += P.my[0]; r1 += P.my[1]; r2 += P.my[2]; r3 += P.my[3];
        }
    }
}

// General setup of one pair (any pitch, any magnitude): 32-bit planes with every value range-checked in int64
// (span_plane) when the tet's lattice bbox is < 2^15 per axis and g is a power of two; anything else, or plane
// values that do not fit int32 on the pair's box, goes to the int64 large path.  Out of line: setup_pair's fast
// path is what nearly every pair of the BASELINE workloads takes.
__device__ __noinline__ bool setup_general(const Params& p, const Tet q, const TileGeo& g, u32 box, int* rec) {
    const int x0 = box & 31, y0 = (box >> 10) & 31, y1 = (box >> 15) & 31, z0 = (box >> 20) & 31, z1 = (box >> 25) & 31;
    const int x1 = (box >> 5) & 31;
    const int ny = y1 - y0 + 1, nz = z1 - z0 + 1, nrows = ny * nz;
    const int lox = min(min(q.ax, q.bx), min(q.cx, q.dx)), hix = max(max(q.ax, q.bx), max(q.cx, q.dx));
    const int loy = min(min(q.ay, q.by), min(q.cy, q.dy)), hiy = max(max(q.ay, q.by), max(q.cy, q.dy));
    const int loz = min(min(q.az, q.bz), min(q.cz, q.dz)), hiz = max(max(q.az, q.bz), max(q.cz, q.dz));
    bool ok = (((hix - lox) | (hiy - loy) | (hiz - loz)) < 32768) && (p.g_shift >= 0);
    int nlo = 0;
    if (ok) {
        const int ux = q.bx - q.ax, uy = q.by - q.ay, uz = q.bz - q.az;
        const int vx = q.cx - q.ax, vy = q.cy - q.ay, vz = q.cz - q.az;
        const int wx = q.dx - q.ax, wy = q.dy - q.ay, wz = q.dz - q.az;
        // N_b = v x w, N_c = u x w, N_d = u x v, N_a = (v-u) x (w-u) = N_b - N_c + N_d
        const int nbx = vy * wz - vz * wy, nby = vz * wx - vx * wz, nbz = vx * wy - vy * wx;
        const int ncx = uy * wz - uz * wy, ncy = uz * wx - ux * wz, ncz = ux * wy - uy * wx;
        const int ndx = uy * vz - uz * vy, ndy = uz * vx - ux * vz, ndz = ux * vy - uy * vx;
        const int nax = (int)((u32)nbx - (u32)ncx + (u32)ndx), nay = (int)((u32)nby - (u32)ncy + (u32)ndy);
        const int naz = (int)((u32)nbz - (u32)ncz + (u32)ndz);
        const i64 det = (i64)ux * nbx + (i64)uy * nby + (i64)uz * nbz;  // 6V = u.(v x w)
        if (det == 0) {  // degenerate (G2): contributes nothing.  (K1 culls these; the fused lattice path meets them here)
            null_record(rec, g.img_saddr);
            return false;
        }
        const int s = det > 0 ? 1 : -1;
        // sigma = (s, -s, s, -s): F = (s*D_a, -s*D_b, s*D_c, -s*D_d) >= 0 inside
        const int arx = q.ax - g.p0x, ary = q.ay - g.p0y, arz = q.az - g.p0z;
        const int brx = q.bx - g.p0x, bry = q.by - g.p0y, brz = q.bz - g.p0z;
        // m_x = -sigma*N_x*sx > 0  <=>  lo-type
        const bool l0 = s * nax < 0, l1 = s * nbx > 0, l2 = s * ncx < 0, l3 = s * ndx > 0;
        nlo = (int)l0 + (int)l1 + (int)l2 + (int)l3;
        const int pos0 = l0 ? 0 : nlo;
        const int pos1 = l1 ? (int)l0 : nlo + (int)!l0;
        const int pos2 = l2 ? (int)l0 + (int)l1 : nlo + (int)!l0 + (int)!l1;
        const int pos3 = l3 ? nlo - 1 : 3;
        ok = span_plane(p, rec, pos0, s * nax, s * nay, s * naz, brx, bry, brz, x0, y0, z0, ny, nz) && ok;
        ok = span_plane(p, rec, pos1, -s * nbx, -s * nby, -s * nbz, arx, ary, arz, x0, y0, z0, ny, nz) && ok;
        ok = span_plane(p, rec, pos2, s * ncx, s * ncy, s * ncz, arx, ary, arz, x0, y0, z0, ny, nz) && ok;
        ok = span_plane(p, rec, pos3, -s * ndx, -s * ndy, -s * ndz, arx, ary, arz, x0, y0, z0, ny, nz) && ok;
    }
    if (!ok) {  // int64 planes for the large path, computed here (one thread per pair) rather than by a whole warp
        if (six_volume(q) == 0) {
            null_record(rec, g.img_saddr);
            return false;
        }
        large_record(p, q, g, box, rec);
        return true;
    }
    // nlo == 0 or 4 cannot happen for a non-degenerate tet (the four sigma*N sum to zero and planes with
    // N_x == 0 count as hi-type); such a record is made to draw nothing: one row, x1' = -2
    const bool valid = nlo >= 1 && nlo <= 3;
    *reinterpret_cast<int4*>(rec) = make_int4(x0 + 1, valid ? x1 - x0 : -2, ny, valid ? nrows : 1);
    *reinterpret_cast<int4*>(rec + 4) =
        make_int4((int)(g.img_saddr + 4u * (u32)(z0 * g.img_stride + y0)), (int)((65536u + ny - 1) / ny),
                  nlo >= 2 ? (1 << 30) : -(1 << 30), nlo == 3 ? (1 << 30) : -(1 << 30));
    return true;
}

// inv in [2^32/a, (2^32/a)(1 + 2^-19) + 1) for 4 <= a < 2^31, never below 2^32/a: a (rounded DOWN to float) through
// rcp.approx (relative error <= 2^-23) times 2^32 (1 + 2^-20), rounded up.  span_bound only needs "not below, and
// relatively within 2^-18" (see there); a wrong bit cannot come from here, the integer check decides.
__device__ __forceinline__ int recip_up(u32 a) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(__uint2float_rd(a)));
    return (int)__float2uint_ru(r * 4294971392.0f);  // 2^32 + 2^12
}

// One plane of the FAST path.  N = the face normal as Theorem 1 orders it (not yet signed), sig = +-1 its sign
// sigma, (rx,ry,rz) = Q - P with P the centre of the box-origin voxel.  With t = sign(N_x) != 0:
//   hi-type <=> sigma*N_x > 0 <=> t == sigma;  stored m = -sigma*N*s (hi) = +sigma*N*s (lo) = -t*N*s in both cases;
//   W = t*N.(Q-P):  Q0 = floor(W/g) (hi: G itself)  or  -floor(-W/g) - 1 = floor((W-1)/g) (lo: -G - 1).
// c4 = -4*s_a folds the sign and the scale by 4 into the pitch ratio.  All values fit int32 (setup_pair's test).
__device__ __forceinline__ void fast_plane(const Params& p, int* rec, int pos, bool lo, int nx, int ny, int nz, int rx,
                                           int ry, int rz) {
    const int t = (nx >> 31) | 1;
    const int ax = abs(nx), by = ny * t, bz = nz * t;
    const i64 W = (i64)ax * rx + (i64)by * ry + (i64)bz * rz - (lo ? 1 : 0);
    const int q0 = (int)(W >> p.g_shift);
    const int mx = ax * p.c4x;  // <= -4
    *reinterpret_cast<int4*>(rec + 8 + 4 * pos) = make_int4(mx, by * p.c4y, bz * p.c4z, q0 << 2);
    rec[24 + pos] = recip_up((u32)(-mx));
}

// M with floor(rr*M / 2^16) == rr / ny for all 0 <= rr < 1024, 1 <= ny <= 32: any M in [2^16/ny, 2^16/ny + 2) will do
// (the excess rr*(M - 2^16/ny)/2^16 stays below 1/ny); floor(2^16/ny) + 1 is one, and the float quotient cannot miss the
// floor: 2^16/ny is exact for powers of two and at least 1/32 away from an integer otherwise.
__device__ __forceinline__ int div_magic(int ny) { return __float2int_rz(__fdividef(65536.0f, (float)ny)) + 1; }

// closed voxel-index range of the centres h*i + h/2 inside [lo, hi]  (not clamped)
template <bool POW2>
__device__ __forceinline__ void centre_range(int lo, int hi, int h, int sh, int& i0, int& i1) {
    if (POW2) {
        i0 = -((h - 2 * lo) >> sh);  // ceil((2lo - h) / 2h)
        i1 = (2 * hi - h) >> sh;
    } else {
        i0 = -floor_div_i(h - 2 * lo, 2 * h);
        i1 = floor_div_i(2 * hi - h, 2 * h);
    }
}

// thread-per-(tet,tile) setup.  The pair's local box (the tet's closed voxel bbox clipped to the tile) comes first;
// an empty box or a degenerate tet gives a record that draws nothing (the binning passes never produce such pairs,
// the fused lattice path does).  FAST path (POW2: every pitch and g a power of two): when
//     24*dx*dy*dz/g + 16*max(dy*dz*sx, dx*dz*sy, dx*dy*sz) < 2*10^9   and   dx,dy,dz < 2^15   (d = lattice bbox extent)
// every stored value fits int32 with room to spare and no per-plane range check is needed:
//   |N_x| <= 2 dy dz (etc.), so |m| = 4|N|s <= 8 d d s;  for every sample P of the box (a point of the tet's bbox)
//   |sigma*N.(Q-P)| <= 6 dx dy dz, so every row value |r| <= 4 (6 dx dy dz / g + 1);  span_bound forms r and r - a*c0
//   with a*|c0| <= |r| (1 + 2^-18) + a: all below 2^31 under the test (float, evaluated with 7% of slack; it only
//   picks the path, both paths are exact).
// Planes with N_x == 0 (row gates) and everything that fails the test take setup_general.
// the four vertices of a tet: one 16-byte load each from K0's packed copy (fused lattice path), else 3 x 4 bytes
template <bool V4>
__device__ __forceinline__ Tet gather_tet(const Params& p, int4 id) {
    VOX_CHECK(id.x >= 0 && id.x < p.V && id.y >= 0 && id.y < p.V && id.z >= 0 && id.z < p.V && id.w >= 0 && id.w < p.V, CK_K4_VERT);
    Tet q;
    if (V4) {
        const int4 a = __ldg(p.verts4 + id.x), b = __ldg(p.verts4 + id.y), c = __ldg(p.verts4 + id.z), d = __ldg(p.verts4 + id.w);
        q.ax = a.x; q.ay = a.y; q.az = a.z; q.bx = b.x; q.by = b.y; q.bz = b.z;
        q.cx = c.x; q.cy = c.y; q.cz = c.z; q.dx = d.x; q.dy = d.y; q.dz = d.z;
    } else {
        const int32_t* v = p.verts;
        q.ax = __ldg(v + 3 * (i64)id.x); q.ay = __ldg(v + 3 * (i64)id.x + 1); q.az = __ldg(v + 3 * (i64)id.x + 2);
        q.bx = __ldg(v + 3 * (i64)id.y); q.by = __ldg(v + 3 * (i64)id.y + 1); q.bz = __ldg(v + 3 * (i64)id.y + 2);
        q.cx = __ldg(v + 3 * (i64)id.z); q.cy = __ldg(v + 3 * (i64)id.z + 1); q.cz = __ldg(v + 3 * (i64)id.z + 2);
        q.dx = __ldg(v + 3 * (i64)id.w); q.dy = __ldg(v + 3 * (i64)id.w + 1); q.dz = __ldg(v + 3 * (i64)id.w + 2);
    }
    return q;
}

struct LocalBox {
    int x0, x1, y0, y1, z0, z1;  // tile-local closed voxel box, empty if any lower bound exceeds its upper bound
    int dx, dy, dz;              // extent of the tet's lattice bbox
};
// the tet's closed voxel bbox (same rounding as K1's axis_range) clipped to the tile
template <bool POW2>
__device__ __forceinline__ bool local_box(const Params& p, const TileGeo& g, const Tet& q, LocalBox& B) {
    const int lox = min(min(q.ax, q.bx), min(q.cx, q.dx)), hix = max(max(q.ax, q.bx), max(q.cx, q.dx));
    const int loy = min(min(q.ay, q.by), min(q.cy, q.dy)), hiy = max(max(q.ay, q.by), max(q.cy, q.dy));
    const int loz = min(min(q.az, q.bz), min(q.cz, q.dz)), hiz = max(max(q.az, q.bz), max(q.cz, q.dz));
    centre_range<POW2>(lox, hix, p.hx, p.qx, B.x0, B.x1);
    centre_range<POW2>(loy, hiy, p.hy, p.qy, B.y0, B.y1);
    centre_range<POW2>(loz, hiz, p.hz, p.qz, B.z0, B.z1);
    B.x0 = max(B.x0 - g.X0, 0); B.x1 = min(B.x1 - g.X0, 31);  // nx % 32 == 0: the tile's 32 columns lie inside the grid
    B.y0 = max(B.y0 - g.Y0, 0); B.y1 = min(B.y1 - g.Y0, g.ymax);
    B.z0 = max(B.z0 - g.Z0, 0); B.z1 = min(B.z1 - g.Z0, g.zmax);
    B.dx = hix - lox; B.dy = hiy - loy; B.dz = hiz - loz;
    return (B.x0 <= B.x1) & (B.y0 <= B.y1) & (B.z0 <= B.z1);
}

template <bool POW2, bool V4>
__device__ __forceinline__ bool setup_pair(const Params& p, const TileGeo& g, int4 id, int* rec) {
    const Tet q = gather_tet<V4>(p, id);
    LocalBox B;
    const bool hit = local_box<POW2>(p, g, q, B);
    const int x0 = B.x0, x1 = B.x1, y0 = B.y0, y1 = B.y1, z0 = B.z0, z1 = B.z1;
    VOX_CHECK(!hit || (x0 >= 0 && x1 <= 31 && y0 >= 0 && y1 <= g.ymax && z0 >= 0 && z1 <= g.zmax && g.ymax <= 31 && g.zmax <= 31), CK_K4_BOX);
    if (!hit) {
        null_record(rec, g.img_saddr);
        return false;
    }
    const int dx = B.dx, dy = B.dy, dz = B.dz;
    bool fast = POW2 && ((dx | dy | dz) < 32768);
    if (fast) {
        const float fx = (float)dx, fy = (float)dy, fz = (float)dz;
        const float fyz = fy * fz;
        fast = fx * fyz * p.fit_vol + fmaxf(fmaxf(fyz * p.fit_ax, fx * fz * p.fit_ay), fx * fy * p.fit_az) < 2.0e9f;
    }
    if (fast) {
        const int ux = q.bx - q.ax, uy = q.by - q.ay, uz = q.bz - q.az;
        const int vx = q.cx - q.ax, vy = q.cy - q.ay, vz = q.cz - q.az;
        const int wx = q.dx - q.ax, wy = q.dy - q.ay, wz = q.dz - q.az;
        // N_b = v x w, N_c = u x w, N_d = u x v, N_a = (v-u) x (w-u) = N_b - N_c + N_d   (all < 2^31: d < 2^15)
        const int nbx = vy * wz - vz * wy, nby = vz * wx - vx * wz, nbz = vx * wy - vy * wx;
        const int ncx = uy * wz - uz * wy, ncy = uz * wx - ux * wz, ncz = ux * wy - uy * wx;
        const int ndx = uy * vz - uz * vy, ndy = uz * vx - ux * vz, ndz = ux * vy - uy * vx;
        const int nax = nbx - ncx + ndx, nay = nby - ncy + ndy, naz = nbz - ncz + ndz;
        const i64 det = (i64)ux * nbx + (i64)uy * nby + (i64)uz * nbz;  // 6V = u.(v x w)
        if (det == 0) {  // degenerate (G2): contributes nothing
            null_record(rec, g.img_saddr);
            return false;
        }
        if ((nax != 0) & (nbx != 0) & (ncx != 0) & (ndx != 0)) {
            const int s = det > 0 ? 1 : -1;
            // sigma = (s, -s, s, -s);  lo-type <=> sign(N_x) != sigma
            const bool l0 = (nax ^ s) < 0, l1 = (nbx ^ s) >= 0, l2 = (ncx ^ s) < 0, l3 = (ndx ^ s) >= 0;
            const int nlo = (int)l0 + (int)l1 + (int)l2 + (int)l3;  // 1..3: the four sigma*N sum to zero
            const int pos0 = l0 ? 0 : nlo;
            const int pos1 = l1 ? (int)l0 : nlo + (int)!l0;
            const int pos2 = l2 ? (int)l0 + (int)l1 : nlo + (int)!l0 + (int)!l1;
            const int pos3 = l3 ? nlo - 1 : 3;
            // Q - P, P = centre of the box-origin voxel;  B - P = (A - P) + u
            const int arx = q.ax - g.p0x - p.hx * x0, ary = q.ay - g.p0y - p.hy * y0, arz = q.az - g.p0z - p.hz * z0;
            fast_plane(p, rec, pos0, l0, nax, nay, naz, arx + ux, ary + uy, arz + uz);
            fast_plane(p, rec, pos1, l1, nbx, nby, nbz, arx, ary, arz);
            fast_plane(p, rec, pos2, l2, ncx, ncy, ncz, arx, ary, arz);
            fast_plane(p, rec, pos3, l3, ndx, ndy, ndz, arx, ary, arz);
            const int ny = y1 - y0 + 1;
            *reinterpret_cast<int4*>(rec) = make_int4(x0 + 1, x1 - x0, ny, ny * (z1 - z0 + 1));
            *reinterpret_cast<int4*>(rec + 4) =
                make_int4((int)(g.img_saddr + 4u * (u32)(z0 * g.img_stride + y0)), div_magic(ny),
                          nlo >= 2 ? (1 << 30) : -(1 << 30), nlo == 3 ? (1 << 30) : -(1 << 30));
            return true;
        }
    }
    return setup_general(p, q, g, pack_box(x0, x1, y0, y1, z0, z1), rec);
}

// b = max{x : Q(x) >= 0} for Q(x) = r - a*x (mx = -a, a >= 4), whenever 0 <= r and that b is below 2^18; some value
// >= 2^18 - 1 when it is not (such a bound does not bind: x' <= 31); some b <= -1 when r < 0.
// inv in [2^32/a, (2^32/a)(1 + 2^-19) + 1) (exact ceil from span_plane, or recip_up): c0 = floor(r*inv/2^32) >= B =
// floor(r/a), and c0 <= B + 1 when r/a < 2^18 (the excess is below r/a * 2^-19 + r/2^32 < 1); for r < 0, c0 <= -1.
// The INTEGER value Q(c0) decides.  |a*c0| <= |r| (1 + 2^-18) + a < 2^31 (guaranteed at setup), so nothing wraps.
__device__ __forceinline__ int span_bound(int r, int mx, int inv) {
    const int c0 = __mulhi(r, inv);
    const int v = r + mx * c0;
    return c0 + (v >> 31);
}

// ------------------------------------------------------------------------------------------
// Row-flattened walk.  The rows of a batch of NT (tet,tile) pairs are laid end to end and dealt out in equal
// runs: thread i draws rows [i*R, (i+1)*R) of the batch, whichever pairs they belong to, stepping to the next
// pair's record when one ends.  Every lane is busy whatever the pairs' sizes are (a pair clipped to 9 rows used
// to occupy a whole warp for one pass), and the four warps of the CTA finish together.
// ------------------------------------------------------------------------------------------
struct LaneRec {
    int4 A;               // x0+1, x1-x0, ny, nrows
    int4 B;               // saddr, magic, c1, c2
    int4 P0, P1, P2, P3;  // plane slots: mx, my, mz, g0
    int4 IV;
};

__device__ __forceinline__ int4 lds128(u32 saddr) {
    int4 v;
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
    return v;
}
// (by shared-memory byte address: the walk keeps the address of its current record in a register and steps it,
//  instead of rebuilding it from the record index at every pair boundary)
__device__ __forceinline__ void lane_load(u32 rec_saddr, LaneRec& L) {
    L.A = lds128(rec_saddr);
    L.B = lds128(rec_saddr + 16);
    L.P0 = lds128(rec_saddr + 32);
    L.P1 = lds128(rec_saddr + 48);
    L.P2 = lds128(rec_saddr + 64);
    L.P3 = lds128(rec_saddr + 80);
    L.IV = lds128(rec_saddr + 96);
}

// one row rr of the pair held in L: the four exact bounds, the span, one OR into the tile image
__device__ __forceinline__ void lane_row(const LaneRec& L, int rr, int img_stride, u32 img_lo, u32 img_hi) {
    const int zz = (int)(((u32)rr * (u32)L.B.y) >> 16);
    const int yy = rr - zz * L.A.z;
    const int b0 = span_bound(L.P0.w + L.P0.y * yy + L.P0.z * zz, L.P0.x, L.IV.x);
    const int b1 = span_bound(L.P1.w + L.P1.y * yy + L.P1.z * zz, L.P1.x, L.IV.y);
    const int b2 = span_bound(L.P2.w + L.P2.y * yy + L.P2.z * zz, L.P2.x, L.IV.z);
    const int b3 = span_bound(L.P3.w + L.P3.y * yy + L.P3.z * zz, L.P3.x, L.IV.w);
    // planes are stored lo-types first: slot 0 is always lo, slot 3 always hi; |b| < 2^30
    // lo-type (c = +2^30): min(b,c) = b joins the lower bounds, max(b,c) = c is no upper bound; hi-type the reverse
    const int l1 = min(b1, L.B.z), u1 = max(b1, L.B.z);
    const int l2 = min(b2, L.B.w), u2 = max(b2, L.B.w);
    const int lower = max(max(-1, b0), max(l1, l2));  // (first solid x') - 1, x' = x - x0
    const int upper = min(min(L.A.y, b3), min(u1, u2));
    const int n = upper - lower;
    const u32 saddr = (u32)L.B.x + 4u * (u32)(zz * img_stride + yy);
    VOX_CHECK(rr >= 0 && rr < L.A.w && yy >= 0 && yy < L.A.z && zz >= 0 && zz <= 31, CK_K4_ROWS);
    VOX_CHECK(saddr >= img_lo && saddr < img_hi && (saddr & 3u) == 0, CK_K4_ROWADDR);
    // branch-free: the word is a mask of max(n, 0) bits from bit lower + 1 + x0 (BMSK); n <= 0 gives 0 and the OR is a no-op
    const int width = max(n, 0), pos = lower + L.A.x;
    asm volatile(
        "{\n\t.reg .b32 m;\n\t"
        "bmsk.clamp.b32 m, %1, %2;\n\t"
        "red.shared.or.b32 [%0], m;\n\t}"
        ::"r"(saddr), "r"(pos), "r"(width)
        : "memory");
}

template <int NT, bool SPARSE>
__device__ __forceinline__ void tile_epilogue(const Params& p, const u32* img, int img_stride, u32 b, u32 bx, u32 m,
                                              int Y0, int Z0, u32* __restrict__ bits, u32* __restrict__ hdr,
                                              const SparseOut& so, int tid) {
    const int TY = 1 << p.ty_log;
    const int rows = 1 << (p.ty_log + p.tz_log);
    if (!SPARSE) {
        // word of row (y,z) = tile base + (z*ny + y)*wpr: the row offset fits 32 bits (z,y < 32, ny <= 32768, wpr <= 1024)
        u32* base = bits + (((size_t)m * p.nz + Z0) * p.ny + Y0) * p.wpr + bx;
        const int ylim = p.ny - Y0, zlim = p.nz - Z0;
        for (int i = tid; i < rows; i += NT) {
            const int z = i >> p.ty_log, y = i & (TY - 1);
            if (y < ylim && z < zlim) {
                VOX_CHECK((((size_t)m * p.nz + Z0 + z) * p.ny + Y0 + y) * p.wpr + bx < (size_t)p.batch * p.nz * p.ny * p.wpr, CK_K4_STORE);
                base[(u32)(z * p.ny + y) * (u32)p.wpr] = img[z * img_stride + y];
            }
        }
        return;
    }
    // classify over the rows that lie inside the grid (ragged last tiles)
    __shared__ u32 s_slot;
    u32 all = 0xFFFFFFFFu, any = 0u;
    for (int i = tid; i < rows; i += NT) {
        const int z = i >> p.ty_log, y = i & (TY - 1);
        if (Y0 + y < p.ny && Z0 + z < p.nz) {
            const u32 w = img[z * img_stride + y];
            all &= w;
            any |= w;
        }
    }
    const int is_full = __syncthreads_and(all == 0xFFFFFFFFu);
    const int is_any = __syncthreads_or(any != 0u);
    if (!is_any || is_full) {
        if (tid == 0) {
            so.table[b] = is_full ? TILE_FULL : TILE_EMPTY;
            if (is_full) atomicAdd(hdr + H_FULL, 1u);
        }
        return;
    }
    if (tid == 0) {
        const u32 slot = atomicAdd(hdr + H_MIXED, 1u);
        s_slot = slot;
        so.table[b] = slot < so.cap ? slot + 1u : TILE_DROPPED;
        if (slot >= so.cap) hdr[H_PAYLOAD_OVERFLOW] = 1;
    }
    __syncthreads();
    const u32 slot = s_slot;
    if (slot >= so.cap) return;
    u32* dst = so.payload + (size_t)slot * rows;
    for (int i = tid; i < rows; i += NT) {
        const int z = i >> p.ty_log, y = i & (TY - 1);
        const bool in = (Y0 + y < p.ny) && (Z0 + z < p.nz);
        dst[i] = in ? img[z * img_stride + y] : 0u;
    }
}
