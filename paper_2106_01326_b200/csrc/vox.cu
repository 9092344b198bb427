// vox.cu -- B200 (sm_100a) tetrahedral-mesh -> solid-binary-voxel hot path.
//
// Kernels:
//   K1 k1_count    per-tet voxel bbox -> tile range, sliver/degenerate cull, per-tile histogram
//   K2 k2_scan     exclusive scan of the tile counts (+ cursors, totals)
//   K3 k3_scatter  tet ids into per-tile lists
//   K4 k4_flat     one CTA per 32 x TY x TZ tile: exact integer edge functions of
//                  Theorem 1, one exact x-span per row, row words formed on
//                  chip, tile image stored once (no global atomics on the grid)
//   K5 (inside K4) large-tet path: exact tile classification + int64 span rows / 64-bit ballot rasteriser
//
// Exactness: inside(P) <=> four affine functions G_k(P) >= 0, each an exact integer
// (DESIGN.md "Arithmetic").  No floating point decides a bit.
#include "../../include/vox.h"

#include <cuda_runtime.h>
#include <pthread.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

typedef long long i64;
typedef unsigned long long u64;
typedef unsigned int u32;

// ------------------------------------------------------------------------------------------
// host context
// ------------------------------------------------------------------------------------------
struct Params {
    const int32_t* verts;
    const int4* tets;
    const i64* off;  // device, [batch+1] or NULL
    const int4* verts4;  // fused lattice path: K0's 16-byte copy of the vertices (x, y, z, 0) in the workspace, else NULL
    const unsigned char* keep;  // lattice input (vox_lattice): bit q of keep[cell] = tet q of the cell is present
    int lcx, lcy, lcz;          // cells per axis of the lattice input; lcx == 0: explicit tets
    int fused;                  // lattice input takes the fused path (lattice_fused)
    i64 T;
    i64 V;
    int batch;
    int nx, ny, nz;
    int hx, hy, hz;      // pitch per axis
    int qx, qy, qz;      // log2(2h) per axis, or -1 when 2h is not a power of two
    int lim_x, lim_y, lim_z;  // (2^30 - 1) / (h/g): largest |N| component whose scaled coefficient fits
    int g, g_shift;      // gcd of the pitches; log2(g) or -1
    int sx, sy, sz;      // h / g
    int c4x, c4y, c4z;   // -4 * (h / g): sign and scale of a stored plane coefficient (setup_pair's fast path)
    int pow2;            // every 2h and g is a power of two: shifts instead of divisions
    int grid3;           // K4 is launched as a 3-D grid (nbx, nby, nbz*batch) rather than 1-D over the tiles
    float fit_vol, fit_ax, fit_ay, fit_az;  // setup_pair's int32 fit test: 24/g, 16*sx, 16*sy, 16*sz
    int ty_log, tz_log;  // tile = 32 x (1<<ty_log) x (1<<tz_log) voxels
    int nbx, nby, nbz;   // tiles per axis
    int wpr;             // words per grid row = nx/32
    u32 NB;              // tiles in the batch
    u32 cap;             // capacity of the pair list
    int ex, ey, ez;
};

struct SparseOut {
    u32* table;    // [NB]; NULL = dense output
    u32* payload;  // [cap][TZ][TY]
    u32 cap;       // payload capacity in tiles
};

struct vox_ctx {
    bool tile_user;      // tile fixed by vox_set_tile (or by a pipe): vox_tets does not re-pick it
    Params p;
    SparseOut sparse;    // set for the duration of vox_run_sparse only
    bool have_tets;
    i64 pairs_planned;  // -1 = unknown
    int variant;
    int tm_slots;        // per-kernel timing ring (0 = off)
    int tm_next;
    cudaEvent_t* tm_ev;  // [tm_slots][TM_EV]
    char err[256];
};
enum { TM_EV = 5 };  // before memset/K1, after K1, after K2, after K3, after K4

enum { HDR_WORDS = 64 };
// header words
enum { H_TOTAL = 0, H_OVERFLOW = 1, H_CULLED = 2, H_LARGE = 3, H_NONEMPTY = 4, H_BAD = 5, H_TOTAL_HI = 6,
       H_MIXED = 7, H_FULL = 8, H_PAYLOAD_OVERFLOW = 9, H_NBIG = 10 };
// tets whose tile range exceeds BIG_TILES are not binned by their own thread: K1 lists them and K2's CTA
// (1024 threads) counts and scatters their tiles
enum { BIG_TILES = 64, BIG_CAP = 4096, RANGE_BIG = 0x40000000 };
// sparse tile table codes (include/vox.h)
#define TILE_EMPTY 0u
#define TILE_FULL 0xFFFFFFFFu
#define TILE_DROPPED 0xFFFFFFFEu

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// Checked build (-DVOX_CHECKS, libvox_checked.so): every index the kernels form is tested before it is used and the
// first violated check's code is kept in g_check (vox_debug_check_status).  compute-sanitizer is closed on this
// pool (profiles/r02_sanitizers.md): these bounds checks, run under the parity suite's small cases, stand in for
// memcheck; the barrier structure that stands in for racecheck is written out there as well.  The normal build
// compiles none of it.
#ifdef VOX_CHECKS
__device__ unsigned int g_check = 0;
#define VOX_CHECK(cond, code)                         \
    do {                                              \
        if (!(cond)) atomicCAS(&g_check, 0u, (unsigned)(code)); \
    } while (0)
#else
#define VOX_CHECK(cond, code) do { } while (0)
#endif
enum {  // check codes
    CK_K1_TILE = 101, CK_K1_VERT = 102, CK_K2_TILE = 201, CK_K3_TILE = 301, CK_K3_RANGE = 302,
    CK_K4_LIST = 401, CK_K4_VERT = 402, CK_K4_BOX = 403, CK_K4_ROWADDR = 404, CK_K4_RECIDX = 405, CK_K4_QUEUE = 406,
    CK_K4_CELL = 407, CK_K4_ROWS = 408, CK_K4_STORE = 409, CK_K4_LARGEBOX = 410, CK_K0_VERT = 501
};

// kernels launched by this library in this process (vox_kernel_launches: bench.py's gpu_launches)
static unsigned long long g_launches = 0;
static inline void count_launch() { __atomic_fetch_add(&g_launches, 1ull, __ATOMIC_RELAXED); }

struct WsLayout {
    size_t hdr, slab, counts, cursor, big, range, list, fixed_end;
};
// fused lattice path: per mesh 2 * ((cx+1) + (cy+1) + (cz+1)) ints of vertex-plane bounds (k0_slabs), else nothing
// (the binned paths keep the layout a pipe sized for them)
static size_t slab_ints(const Params& p) {
    return p.fused ? (size_t)p.batch * 2 * ((size_t)p.lcx + p.lcy + p.lcz + 3) : 0;
}
static WsLayout ws_layout(const Params& p) {
    WsLayout L;
    size_t o = 0;
    L.hdr = o;
    o = align256(o + HDR_WORDS * 4);
    L.slab = o;  // (header, slabs and counts are adjacent: one memset clears them)
    o = align256(o + slab_ints(p) * 4);
    L.counts = o;
    o = align256(o + ((size_t)p.NB + 1) * 4);
    L.cursor = o;
    o = align256(o + ((size_t)p.NB + 1) * 4);
    L.big = o;
    o = align256(o + (size_t)BIG_CAP * 4);
    L.range = o;
    o = align256(o + (size_t)(p.T > 0 ? p.T : 1) * 8);
    L.list = o;
    L.fixed_end = o;
    return L;
}

// ------------------------------------------------------------------------------------------
// device helpers: integer geometry
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int floor_div_i(int a, int b) {  // b > 0
    int q = a / b;
    int r = a - q * b;
    return (r < 0) ? q - 1 : q;
}
// floor(a / 2h): an arithmetic shift when 2h is a power of two (sh = log2(2h)), else a division
__device__ __forceinline__ int floor_div_2h(int a, int h, int sh) {
    return (sh >= 0) ? (a >> sh) : floor_div_i(a, 2 * h);
}
__device__ __forceinline__ i64 floor_div_l(i64 a, i64 b) {  // b > 0
    i64 q = a / b;
    i64 r = a - q * b;
    return (r < 0) ? q - 1 : q;
}

struct Tet {
    int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
};

// Lattice input (include/vox.h "vox_lattice"): tet t = 6*cell + q of cell (i,j,k) walks from the cell's low corner
// along the axes of the q-th permutation of (x,y,z) in lexicographic order; vertex id = (i*(cy+1) + j)*(cz+1) + k.
__device__ __forceinline__ int4 lattice_ids(const Params& p, i64 t64) {
    // 32-bit arithmetic throughout: T = 6 * cells * batch <= 0xFFFFFFF0 (vox_lattice)
    const u32 t = (u32)t64;
    const int q = (int)(t % 6u);
    u32 c = t / 6u;
    const u32 cells = (u32)p.lcx * (u32)p.lcy * (u32)p.lcz;
    const int mesh = (p.batch == 1) ? 0 : (int)(c / cells);  // mesh m owns cells [m*cells, (m+1)*cells) and its own vertex block
    c -= (u32)mesh * cells;
    const int k = (int)(c % (u32)p.lcz);
    c /= (u32)p.lcz;
    const int j = (int)(c % (u32)p.lcy);
    const int i = (int)(c / (u32)p.lcy);
    const int sz = 1, sy = p.lcz + 1, sx = (p.lcy + 1) * (p.lcz + 1);
    const int v0 = mesh * (p.lcx + 1) * sx + (i * (p.lcy + 1) + j) * (p.lcz + 1) + k;
    // permutations of (x,y,z), lexicographic: xyz xzy yxz yzx zxy zyx
    const int a1 = (q < 2) ? sx : (q < 4) ? sy : sz;
    const int a3 = (q == 3 || q == 5) ? sx : (q == 1 || q == 4) ? sy : sz;
    const int a2 = sx + sy + sz - a1 - a3;
    return make_int4(v0, v0 + a1, v0 + a1 + a2, v0 + a1 + a2 + a3);
}

__device__ __forceinline__ Tet load_tet(const Params& p, i64 t) {
    const int4 id = p.lcx ? lattice_ids(p, t) : __ldg(p.tets + t);
    VOX_CHECK(id.x >= 0 && id.x < p.V && id.y >= 0 && id.y < p.V && id.z >= 0 && id.z < p.V && id.w >= 0 && id.w < p.V, CK_K1_VERT);
    const int32_t* v = p.verts;
    Tet q;
    q.ax = __ldg(v + 3 * (i64)id.x); q.ay = __ldg(v + 3 * (i64)id.x + 1); q.az = __ldg(v + 3 * (i64)id.x + 2);
    q.bx = __ldg(v + 3 * (i64)id.y); q.by = __ldg(v + 3 * (i64)id.y + 1); q.bz = __ldg(v + 3 * (i64)id.y + 2);
    q.cx = __ldg(v + 3 * (i64)id.z); q.cy = __ldg(v + 3 * (i64)id.z + 1); q.cz = __ldg(v + 3 * (i64)id.z + 2);
    q.dx = __ldg(v + 3 * (i64)id.w); q.dy = __ldg(v + 3 * (i64)id.w + 1); q.dz = __ldg(v + 3 * (i64)id.w + 2);
    return q;
}

// 6V = det[B-A; C-A; D-A]  (Lemma 1.1)
__device__ __forceinline__ i64 six_volume(const Tet& q) {
    const int ux = q.bx - q.ax, uy = q.by - q.ay, uz = q.bz - q.az;
    const int vx = q.cx - q.ax, vy = q.cy - q.ay, vz = q.cz - q.az;
    const int wx = q.dx - q.ax, wy = q.dy - q.ay, wz = q.dz - q.az;
    // every edge component below 2^15 (the usual case): v x w fits int32, only the final dot product is 64-bit
    const int big = abs(ux) | abs(uy) | abs(uz) | abs(vx) | abs(vy) | abs(vz) | abs(wx) | abs(wy) | abs(wz);
    if (big < 32768) {
        const int cx = vy * wz - vz * wy, cy = vz * wx - vx * wz, cz = vx * wy - vy * wx;
        return (i64)ux * cx + (i64)uy * cy + (i64)uz * cz;
    }
    return (i64)ux * ((i64)vy * wz - (i64)vz * wy) - (i64)uy * ((i64)vx * wz - (i64)vz * wx) + (i64)uz * ((i64)vx * wy - (i64)vy * wx);
}

// closed voxel-index range of centres h*i + h/2 inside [lo, hi], clamped to the grid
__device__ __forceinline__ void axis_range(int a, int b, int c, int d, int h, int sh, int n, int& i0, int& i1) {
    int lo = min(min(a, b), min(c, d));
    int hi = max(max(a, b), max(c, d));
    i0 = -floor_div_2h(h - 2 * lo, h, sh);  // ceil((2lo - h) / 2h)
    i1 = floor_div_2h(2 * hi - h, h, sh);
    i0 = max(i0, 0);
    i1 = min(i1, n - 1);
}

__device__ __forceinline__ int mesh_of(const Params& p, i64 t) {
    if (p.batch == 1) return 0;
    if (p.lcx) return (int)((u32)t / (6u * (u32)p.lcx * (u32)p.lcy * (u32)p.lcz));  // lattice input: equal blocks per mesh
    int lo = 0, hi = p.batch;  // off[lo] <= t < off[hi]
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(p.off + mid) <= t) lo = mid; else hi = mid;
    }
    return lo;
}

// ------------------------------------------------------------------------------------------
// K1: per-tet voxel bbox -> tile range, cull, histogram
// ------------------------------------------------------------------------------------------
#define RANGE_CULLED 0xFFFFFFFFu

__global__ void __launch_bounds__(256) k1_count(Params p, uint2* __restrict__ range, u32* __restrict__ counts,
                                                u32* __restrict__ hdr, u32* __restrict__ big) {
    i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = false, handed = false;
    uint2 r = make_uint2(RANGE_CULLED, 0u);
    int m = 0;
    int b0x = 0, b1x = -1, b0y = 0, b1y = -1, b0z = 0, b1z = -1;
    const bool present = (t < p.T) && (!p.lcx || ((__ldg(p.keep + (u32)t / 6u) >> (int)((u32)t % 6u)) & 1));
    // (lattice input: a tet its cell does not keep gets no range entry -- K3 looks at the keep bit first)
    if (present) {
        Tet q = load_tet(p, t);
        int x0, x1, y0, y1, z0, z1;
        axis_range(q.ax, q.bx, q.cx, q.dx, p.hx, p.qx, p.nx, x0, x1);
        axis_range(q.ay, q.by, q.cy, q.dy, p.hy, p.qy, p.ny, y0, y1);
        axis_range(q.az, q.bz, q.cz, q.dz, p.hz, p.qz, p.nz, z0, z1);
        live = (x0 <= x1) && (y0 <= y1) && (z0 <= z1) && (six_volume(q) != 0);
        if (live) {
            b0x = x0 >> 5; b1x = x1 >> 5;
            b0y = y0 >> p.ty_log; b1y = y1 >> p.ty_log;
            b0z = z0 >> p.tz_log; b1z = z1 >> p.tz_log;
            r.x = (u32)b0x | ((u32)b0y << 10) | ((u32)b0z << 20);
            r.y = (u32)b1x | ((u32)b1y << 10) | ((u32)b1z << 20);
            m = mesh_of(p, t);
            if ((b1x - b0x + 1) * (b1y - b0y + 1) * (b1z - b0z + 1) > BIG_TILES) {  // oversized: hand over to K2
                const u32 slot = atomicAdd(hdr + H_NBIG, 1u);
                if (slot < (u32)BIG_CAP) {
                    big[slot] = (u32)t;
                    r.x |= RANGE_BIG;
                    handed = true;
                }
            }
        }
        range[t] = r;
    }
    unsigned dead = __ballot_sync(0xFFFFFFFFu, present && !live);
    if ((threadIdx.x & 31) == 0 && dead) atomicAdd(hdr + H_CULLED, __popc(dead));
    // warp-aggregated histogram: in step k every live lane names the k-th tile of its range; lanes
    // naming the same tile (neighbouring tets mostly do) are merged into one atomic
    live = live && !handed;
    int cx = b0x, cy = b0y, cz = b0z;
    const int lane = threadIdx.x & 31;
    for (;;) {
        const unsigned act = __ballot_sync(0xFFFFFFFFu, live);
        if (!act) break;
        if (live) {
            const u32 b = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(b < p.NB, CK_K1_TILE);
            const unsigned peers = __match_any_sync(act, b);
            if (lane == __ffs(peers) - 1) atomicAdd(counts + b, (u32)__popc(peers));
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// K2: exclusive scan of counts[0..NB) (single CTA, 4096 counters per pass; NB is at most a few 10^5)
// counts[b] <- offset, counts[NB] <- total, cursor[b] <- offset
// ------------------------------------------------------------------------------------------
// tile b of the idx-th tile of a packed range
__device__ __forceinline__ u32 range_tile(const Params& p, uint2 r, int m, u32 idx) {
    const u32 b0x = r.x & 1023, b0y = (r.x >> 10) & 1023, b0z = (r.x >> 20) & 1023;
    const u32 wx = (r.y & 1023) - b0x + 1, wy = ((r.y >> 10) & 1023) - b0y + 1;
    const u32 dx = idx % wx, rest = idx / wx;
    const u32 dy = rest % wy, dz = rest / wy;
    return ((((u32)m * p.nbz + b0z + dz) * p.nby + b0y + dy) * p.nbx) + b0x + dx;
}
__device__ __forceinline__ u32 range_tiles(uint2 r) {
    const u32 wx = (r.y & 1023) - (r.x & 1023) + 1, wy = ((r.y >> 10) & 1023) - ((r.x >> 10) & 1023) + 1;
    const u32 wz = ((r.y >> 20) & 1023) - ((r.x >> 20) & 1023) + 1;
    return wx * wy * wz;
}

__global__ void __launch_bounds__(1024) k2_scan(Params p, const uint2* __restrict__ range, const u32* __restrict__ big,
                                                u32* __restrict__ list, u32* __restrict__ counts,
                                                u32* __restrict__ cursor, u32* __restrict__ hdr, int scatter_big) {
    const u32 NB = p.NB;
    // oversized tets (K1 listed them): the whole CTA counts their tiles, 1024 at a time
    const u32 nbig = min(hdr[H_NBIG], (u32)BIG_CAP);
    for (u32 e = 0; e < nbig; ++e) {
        const u32 t = big[e];
        const uint2 r = range[t];
        const int m = mesh_of(p, t);
        const u32 n = range_tiles(r);
        for (u32 idx = threadIdx.x; idx < n; idx += 1024u) {
            VOX_CHECK(range_tile(p, r, m, idx) < p.NB, CK_K2_TILE);
            atomicAdd(counts + range_tile(p, r, m, idx), 1u);
        }
    }
    if (nbig) {
        __threadfence();
        __syncthreads();
    }
    // chunks of 4096 counters: one coalesced uint4 per thread, warp shuffle scan, 32 warp partials
    // scanned by warp 0, running carry in 64 bits (a total above 2^32 raises the overflow flag)
    __shared__ u64 s_warp[32];
    __shared__ u64 s_carry;
    __shared__ u32 s_ne[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool vec_ok = ((size_t)counts & 15) == 0 && ((size_t)cursor & 15) == 0;
    if (tid == 0) s_carry = 0;
    u32 ne = 0;
    auto load4 = [&](u32 i) {
        uint4 c = make_uint4(0u, 0u, 0u, 0u);
        if (i + 3 < NB && vec_ok) c = __ldcg(reinterpret_cast<const uint4*>(counts + i));
        else {
            if (i < NB) c.x = __ldcg(counts + i);
            if (i + 1 < NB) c.y = __ldcg(counts + i + 1);
            if (i + 2 < NB) c.z = __ldcg(counts + i + 2);
            if (i + 3 < NB) c.w = __ldcg(counts + i + 3);
        }
        return c;
    };
    uint4 nxt = load4((u32)tid * 4u);
    for (u32 base = 0; base < NB; base += 4096u) {
        const u32 i = base + (u32)tid * 4u;
        const uint4 c = nxt;
        if (base + 4096u < NB) nxt = load4(i + 4096u);  // prefetch the next chunk
        ne += (c.x != 0) + (c.y != 0) + (c.z != 0) + (c.w != 0);
        const u64 mine = (u64)c.x + c.y + c.z + c.w;
        u64 incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        __syncthreads();  // s_warp / s_carry of the previous chunk are consumed
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            const u64 w = s_warp[lane];
            u64 wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const u64 v = __shfl_up_sync(0xFFFFFFFFu, wi, o);
                if (lane >= o) wi += v;
            }
            const u64 carry = s_carry;
            s_warp[lane] = carry + wi - w;  // exclusive offset of each warp, carry included
            __syncwarp();
            if (lane == 31) s_carry = carry + wi;
        }
        __syncthreads();
        const u64 run = s_warp[warp] + incl - mine;
        uint4 o4;
        o4.x = (u32)run;
        o4.y = (u32)(run + c.x);
        o4.z = (u32)(run + c.x + c.y);
        o4.w = (u32)(run + c.x + c.y + c.z);
        if (i + 3 < NB && vec_ok) {
            *reinterpret_cast<uint4*>(counts + i) = o4;
            *reinterpret_cast<uint4*>(cursor + i) = o4;
        } else {
            if (i < NB) { counts[i] = o4.x; cursor[i] = o4.x; }
            if (i + 1 < NB) { counts[i + 1] = o4.y; cursor[i + 1] = o4.y; }
            if (i + 2 < NB) { counts[i + 2] = o4.z; cursor[i + 2] = o4.z; }
            if (i + 3 < NB) { counts[i + 3] = o4.w; cursor[i + 3] = o4.w; }
        }
    }
    for (int o = 16; o; o >>= 1) ne += __shfl_xor_sync(0xFFFFFFFFu, ne, o);
    if (lane == 0) s_ne[warp] = ne;
    __syncthreads();
    if (tid == 0) {
        const u64 total = s_carry;
        counts[NB] = (u32)min(total, (u64)0xFFFFFFFFu);
        hdr[H_TOTAL] = (u32)total;
        hdr[H_TOTAL_HI] = (u32)(total >> 32);
        if (total > 0xFFFFFFFFull) hdr[H_OVERFLOW] = 1;
        u32 s = 0;
        for (int k = 0; k < 32; ++k) s += s_ne[k];
        hdr[H_NONEMPTY] = s;
    }
    if (nbig && scatter_big) {  // scatter the oversized tets (K3 appends the others to the same cursors afterwards)
        __threadfence();
        __syncthreads();
        for (u32 e = 0; e < nbig; ++e) {
            const u32 t = big[e];
            const uint2 r = range[t];
            const int m = mesh_of(p, t);
            const u32 n = range_tiles(r);
            for (u32 idx = threadIdx.x; idx < n; idx += 1024u) {
                const u32 pos = atomicAdd(cursor + range_tile(p, r, m, idx), 1u);
                if (pos < p.cap) list[pos] = t;
                else hdr[H_OVERFLOW] = 1;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// K3: scatter tet ids into the per-tile lists
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k3_scatter(Params p, const uint2* __restrict__ range, u32* __restrict__ cursor,
                                                  u32* __restrict__ list, u32* __restrict__ hdr) {
    i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool live = false;
    int b0x = 0, b0y = 0, b1x = 0, b1y = 0, b1z = 0, cx = 0, cy = 0, cz = 0, m = 0;
    if (t < p.T && (!p.lcx || ((__ldg(p.keep + (u32)t / 6u) >> (int)((u32)t % 6u)) & 1))) {
        const uint2 r = range[t];
        if (r.x != RANGE_CULLED && !(r.x & RANGE_BIG)) {  // (oversized tets were scattered by K2)
            live = true;
            b0x = r.x & 1023; b0y = (r.x >> 10) & 1023; cz = (r.x >> 20) & 1023;
            b1x = r.y & 1023; b1y = (r.y >> 10) & 1023; b1z = (r.y >> 20) & 1023;
            cx = b0x; cy = b0y;
            m = mesh_of(p, t);
        }
    }
    // (tried, round 2: one atomic per (tet, tile) with up to 8 in flight per thread instead of the lockstep aggregation --
    //  2-3.5x slower, 0.15 against 0.072 ms on cfg4, 0.32 against 0.092 on the 10^7-tet mesh: the cursors of a tile are hot
    //  addresses and the number of atomics, not their latency, is what binds)
    // warp-aggregated cursor bump (same stepping as K1): one atomic per distinct tile per step, the lanes of a group
    // take consecutive slots (order inside a tile list is irrelevant: OR).  TWO steps per trip: the kernel is bound by
    // the round trip of the returning atomics, and most tets touch one or two tiles, so the atomics of a lane's next
    // tile are put in flight together with those of its current one.
    const int lane = threadIdx.x & 31;
    const u32 lt = (1u << lane) - 1u;
    for (;;) {
        const unsigned actA = __ballot_sync(0xFFFFFFFFu, live);
        if (!actA) break;
        u32 bA = 0, bB = 0;
        unsigned peersA = 0, peersB = 0;
        bool liveB = false;
        if (live) {
            bA = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(bA < p.NB, CK_K3_TILE);
            peersA = __match_any_sync(actA, bA);
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
            liveB = live;
        }
        const unsigned actB = __ballot_sync(0xFFFFFFFFu, liveB);
        if (liveB) {
            bB = ((((u32)m * p.nbz + cz) * p.nby + cy) * p.nbx) + cx;
            VOX_CHECK(bB < p.NB, CK_K3_TILE);
            peersB = __match_any_sync(actB, bB);
            if (++cx > b1x) {
                cx = b0x;
                if (++cy > b1y) {
                    cy = b0y;
                    live = (++cz <= b1z);
                }
            }
        }
        // both groups' atomics in flight before either result is used
        u32 baseA = 0, baseB = 0;
        if (peersA && lane == __ffs(peersA) - 1) baseA = atomicAdd(cursor + bA, (u32)__popc(peersA));
        if (peersB && lane == __ffs(peersB) - 1) baseB = atomicAdd(cursor + bB, (u32)__popc(peersB));
        if (peersA) {
            baseA = __shfl_sync(peersA, baseA, __ffs(peersA) - 1);
            const u32 pos = baseA + (u32)__popc(peersA & lt);
            if (pos < p.cap) list[pos] = (u32)t;
            else hdr[H_OVERFLOW] = 1;
        }
        if (peersB) {
            baseB = __shfl_sync(peersB, baseB, __ffs(peersB) - 1);
            const u32 pos = baseB + (u32)__popc(peersB & lt);
            if (pos < p.cap) list[pos] = (u32)t;
            else hdr[H_OVERFLOW] = 1;
        }
    }
}

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

// ------------------------------------------------------------------------------------------
// K0 (fused lattice path): one pass over the lattice vertices that
//  (1) records per mesh, axis and vertex plane of the lattice the largest coordinate and the largest
//      (extent - coordinate) over the plane's vertices.  From these a tile finds the index range of the cells whose
//      tets can reach it (k4_flat<.., LATTICE>) -- no per-tet bbox search, no pair list;
//        slab of mesh m: [x: lo'(cx+1) hi(cx+1) | y: lo'(cy+1) hi(cy+1) | z: lo'(cz+1) hi(cz+1)],  lo' = extent - min
//      (zero-initialised by the memset of the header; coordinates lie in [0, extent], so a plain max suffices);
//  (2) writes a 16-byte copy (x, y, z, 0) of every vertex: K4 then gathers a vertex with one LDG.128 instead of three
//      4-byte loads (the gather is what loads the LSU pipe in K4's setup, profiles/r02).
// One CTA per (x plane i, chunk of y rows, mesh); its warps take the chunk's rows in turn, lanes run along z.
// x: registers + warp reduce; y: warp reduce per row; z: shared-memory atomics; one global atomicMax per value and CTA.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k0_slabs(const int32_t* __restrict__ verts, int cx, int cy, int cz, int ex, int ey,
                                                int ez, int jchunk, int* __restrict__ slab, int4* __restrict__ verts4) {
    extern __shared__ int s_z[];  // [cz+1] lo', [cz+1] hi
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = blockIdx.x, m = blockIdx.z;
    const int j0 = blockIdx.y * jchunk, j1 = min(cy + 1, j0 + jchunk);
    int* sl = slab + (size_t)m * 2 * (cx + cy + cz + 3);
    int* xlo = sl, *xhi = sl + cx + 1, *ylo = sl + 2 * (cx + 1), *yhi = ylo + cy + 1, *zlo = ylo + 2 * (cy + 1), *zhi = zlo + cz + 1;
    for (int k = tid; k < 2 * (cz + 1); k += 256) s_z[k] = 0;
    __syncthreads();
    int mxlo = 0, mxhi = 0;
    for (int j = j0 + warp; j < j1; j += 8) {
        int mylo = 0, myhi = 0;
        const size_t v0 = (((size_t)m * (cx + 1) + i) * (cy + 1) + j) * (size_t)(cz + 1);
        const int32_t* row = verts + 3 * v0;
        for (int k = lane; k <= cz; k += 32) {
            const int x = __ldg(row + 3 * k), y = __ldg(row + 3 * k + 1), z = __ldg(row + 3 * k + 2);
            VOX_CHECK(v0 + k < (size_t)gridDim.z * (cx + 1) * (cy + 1) * (cz + 1), CK_K0_VERT);
            verts4[v0 + k] = make_int4(x, y, z, 0);
            mxhi = max(mxhi, x); mxlo = max(mxlo, ex - x);
            myhi = max(myhi, y); mylo = max(mylo, ey - y);
            atomicMax(s_z + k, ez - z);
            atomicMax(s_z + cz + 1 + k, z);
        }
        myhi = __reduce_max_sync(0xFFFFFFFFu, myhi);
        mylo = __reduce_max_sync(0xFFFFFFFFu, mylo);
        if (lane == 0) { atomicMax(yhi + j, myhi); atomicMax(ylo + j, mylo); }
    }
    mxhi = __reduce_max_sync(0xFFFFFFFFu, mxhi);
    mxlo = __reduce_max_sync(0xFFFFFFFFu, mxlo);
    if (lane == 0) { atomicMax(xhi + i, mxhi); atomicMax(xlo + i, mxlo); }
    __syncthreads();
    for (int k = tid; k <= cz; k += 256) { atomicMax(zlo + k, s_z[k]); atomicMax(zhi + k, s_z[cz + 1 + k]); }
}

// ------------------------------------------------------------------------------------------
// K4 kernel.  LATTICE = false: the tile's pairs come from the list the binning passes K1-K3 wrote.
// LATTICE = true (fused lattice path): the tile enumerates its candidate tets itself.  From K0's slabs each of the
// first three warps finds, for one axis, the first and last cell whose vertex planes reach the tile's sample
// centres: every tet that has a sample in the tile lies in that index box (a superset).  The box's cells are dealt
// to the warps in chunks of 32; a lane whose keep bit is set gathers its tet and takes the exact local box
// (local_box, the one setup_pair uses): only the tets that really reach the tile enter the warp's queue (ballot
// compaction), 32 of which are set up per batch on dense lanes.  No K1/K2/K3, no range array, no pair list; the
// price is the box test of the candidates in the rim of the index box.
// ------------------------------------------------------------------------------------------
template <int NT, int MINB, bool SPARSE, bool LATTICE>
__global__ void __launch_bounds__(NT, MINB) k4_flat(const __grid_constant__ Params p, const u32* __restrict__ offsets,
                                                    const u32* __restrict__ list, u32* __restrict__ bits,
                                                    u32* __restrict__ hdr, const __grid_constant__ SparseOut so,
                                                    const int* __restrict__ slab) {
    __shared__ u32 img[32 * (32 + IMG_SKEW)];
    __shared__ __align__(16) int rec[REC_WORDS(NT)];
    __shared__ int s_incl[NT];  // inclusive scan of the pairs' row counts inside each warp's 32 records
    __shared__ int s_wtot[NT / 32];
    __shared__ u32 s_large;
    __shared__ u32 s_wq[LATTICE ? NT / 32 : 1][LATTICE ? 64 : 1];  // per-warp queue of kept candidates: v0 << 3 | q
    __shared__ int s_rng[LATTICE ? 6 : 1];
    __shared__ u32 s_pairs;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NW = NT / 32;
    // tile (bx, by, bz) of mesh m: a 3-D grid (x, y, z*batch) when that fits gridDim (no divisions), else 1-D over tiles
    u32 b, bx, by, bz, m;
    if (p.grid3) {
        bx = blockIdx.x; by = blockIdx.y;
        m = (p.batch == 1) ? 0u : blockIdx.z / (u32)p.nbz;
        bz = blockIdx.z - m * (u32)p.nbz;
        b = ((m * p.nbz + bz) * p.nby + by) * p.nbx + bx;
    } else {
        b = blockIdx.x;
        bx = b % p.nbx;
        u32 rest = b / p.nbx;
        by = rest % p.nby;
        rest /= p.nby;
        bz = rest % p.nbz;
        m = rest / p.nbz;
    }
    const int TY = 1 << p.ty_log, TZ = 1 << p.tz_log;
    TileGeo g;
    g.X0 = bx << 5; g.Y0 = by << p.ty_log; g.Z0 = bz << p.tz_log;
    g.ymax = min(TY, p.ny - g.Y0) - 1;
    g.zmax = min(TZ, p.nz - g.Z0) - 1;
    g.p0x = p.hx * g.X0 + (p.hx >> 1); g.p0y = p.hy * g.Y0 + (p.hy >> 1); g.p0z = p.hz * g.Z0 + (p.hz >> 1);
    g.img_stride = TY + IMG_SKEW;
    g.img_saddr = (u32)__cvta_generic_to_shared(img);
    const u32 rec_saddr = (u32)__cvta_generic_to_shared(rec);
    const int img_stride = g.img_stride;
    const int img_words = img_stride << p.tz_log;
    u32 base = 0, end = 0;
    // LATTICE: candidate index box [ci0, ci0+ni) x [cj0, cj0+nj) x [ck0, ck0+nk), ncand = 6 * cells
    int ci0 = 0, cj0 = 0, ck0 = 0, nj = 1, nk = 1, wq_n = 0;
    u32 ncell = 0, chunk = warp, my_pairs = 0;
    int grp = 0;  // next group of the current chunk (fill stage)
    const u32 cell_base = m * (u32)p.lcx, vert_base = m * (u32)(p.lcx + 1);  // (32-bit: cells and vertices are below 2^31)
    // LATTICE: lane = (cell lane_c of the chunk's five, tet lane_q of the cell's six); tet q walks from the cell's low
    // corner along the axes of the q-th permutation of (x,y,z), lexicographic: xyz xzy yxz yzx zxy zyx (lattice_ids)
    const int lane_c = lane / 6, lane_q = lane - 6 * lane_c;
    const int lat_sy = p.lcz + 1, lat_sx = (p.lcy + 1) * (p.lcz + 1), a123 = lat_sx + lat_sy + 1;
    const int lane_a1 = (lane_q < 2) ? lat_sx : (lane_q < 4) ? lat_sy : 1;
    const int lane_a12 = a123 - ((lane_q == 3 || lane_q == 5) ? lat_sx : (lane_q == 1 || lane_q == 4) ? lat_sy : 1);
    float rnk = 0.f, rnj = 0.f;
    bool small_box = false;
    if (!LATTICE) {
        base = offsets[b];
        end = min(offsets[b + 1], p.cap);
        if (SPARSE && base >= end) {  // no tets: empty tile, nothing else to do
            if (tid == 0) so.table[b] = TILE_EMPTY;
            return;
        }
    } else {
        if (warp < 3) {
            const int c = warp == 0 ? p.lcx : warp == 1 ? p.lcy : p.lcz;  // cells along this warp's axis
            const int* lo = slab + (size_t)m * 2 * (p.lcx + p.lcy + p.lcz + 3) +
                            (warp == 0 ? 0 : warp == 1 ? 2 * (p.lcx + 1) : 2 * (p.lcx + 1) + 2 * (p.lcy + 1));
            const int* hi = lo + c + 1;
            const int E = warp == 0 ? p.ex : warp == 1 ? p.ey : p.ez;
            // the tile's sample centres along this axis: [clo, chi]
            const int clo = warp == 0 ? g.p0x : warp == 1 ? g.p0y : g.p0z;
            const int chi = clo + (warp == 0 ? 31 * p.hx : warp == 1 ? g.ymax * p.hy : g.zmax * p.hz);
            int first = 0x7FFFFFFF, last = -1;
            for (int i0 = 0; i0 < c; i0 += 32) {
                const int i = i0 + lane;
                bool reach = false;
                if (i < c) {  // cell i lies between the vertex planes i and i+1
                    const int cmin = E - max(__ldg(lo + i), __ldg(lo + i + 1)), cmax = max(__ldg(hi + i), __ldg(hi + i + 1));
                    reach = (cmax >= clo) && (cmin <= chi);
                }
                const unsigned bal = __ballot_sync(0xFFFFFFFFu, reach);
                if (bal) {
                    first = min(first, i0 + __ffs(bal) - 1);
                    last = max(last, i0 + 31 - __clz(bal));
                }
            }
            if (lane == 0) { s_rng[2 * warp] = first; s_rng[2 * warp + 1] = last; }
        }
        if (tid == 0) s_pairs = 0;
        __syncthreads();
        ci0 = s_rng[0]; cj0 = s_rng[2]; ck0 = s_rng[4];
        const int ni = max(s_rng[1] - ci0 + 1, 0);
        nj = max(s_rng[3] - cj0 + 1, 0);
        nk = max(s_rng[5] - ck0 + 1, 0);
        ncell = (u32)ni * (u32)nj * (u32)nk;
        small_box = ncell < (1u << 21);
        rnk = 1.0f / (float)max(nk, 1);
        rnj = 1.0f / (float)max(nj, 1);
        if (SPARSE && ncell == 0) {
            if (tid == 0) so.table[b] = TILE_EMPTY;
            return;
        }
    }
    for (int i = tid; i < img_words; i += NT) img[i] = 0;
    if (tid == 0) s_large = 0;
    u32 seen_large = 0;
    for (;;) {
        int n, nr = 0;
        if (!LATTICE) {
            if (base >= end) break;
            __syncthreads();
            n = min((u32)NT, end - base);
            if (tid < n) {
                int* r = rec + rec_off(tid);
                const u32 t = list[base + tid];
                VOX_CHECK((i64)t < p.T && base + tid < p.cap, CK_K4_LIST);
                const int4 id = p.lcx ? lattice_ids(p, t) : __ldg(p.tets + t);
                if (p.pow2) setup_pair<true, false>(p, g, id, r);
                else setup_pair<false, false>(p, g, id, r);
                if (r[6] == 0) atomicAdd(&s_large, 1u);
                nr = r[3];  // >= 1 for every pair: large pairs carry a one-row header that draws nothing
            }
            base += NT;
        } else {
            // fill this warp's queue until it holds a batch's worth.  A chunk is 32 cells of the index box, one per
            // lane: decode the cell, fetch its keep byte (a chunk without kept tets costs just that).  Its candidates
            // are then taken in groups of 5 cells x 6 tets (lane = (lane_c, lane_q), the cell's data by shuffle): a lane
            // whose keep bit is set gathers its tet and takes the exact local box; the tets that reach the tile are
            // appended to the queue.  When the queue is full in mid-chunk the walk stops after group grp and the next
            // batch resumes there (the chunk's decode is simply done again).
            u32* wq = s_wq[warp];
            while (wq_n < 32 && chunk * 32u < ncell) {
                const u32 cell = chunk * 32u + lane;
                u32 kb = 0;
                int v0 = 0;
                if (cell < ncell) {
                    u32 t2, di;
                    if (small_box) {  // exact for cell < 2^21: (cell + 0.5)/nk is at least 0.5/nk away from an integer
                        t2 = (u32)__float2int_rz(((float)cell + 0.5f) * rnk);
                        di = (u32)__float2int_rz(((float)t2 + 0.5f) * rnj);
                    } else {
                        t2 = cell / (u32)nk;
                        di = t2 / (u32)nj;
                    }
                    const u32 i = ci0 + di, j = cj0 + (t2 - di * (u32)nj), k = ck0 + (cell - t2 * (u32)nk);
                    VOX_CHECK(i < (u32)p.lcx && j < (u32)p.lcy && k < (u32)p.lcz, CK_K4_CELL);
                    kb = __ldg(p.keep + (size_t)(((cell_base + i) * p.lcy + j) * p.lcz + k)) & 63u;
                    v0 = (int)(((vert_base + i) * (p.lcy + 1) + j) * (p.lcz + 1) + k);
                }
                const unsigned any = __ballot_sync(0xFFFFFFFFu, kb != 0);
                if (any) {
                    for (; grp < 7; ++grp) {
                        if (((any >> (5 * grp)) & 31u) == 0) continue;  // none of the group's five cells keeps a tet
                        const int src = 5 * grp + lane_c;
                        const u32 kbs = __shfl_sync(0xFFFFFFFFu, kb, src & 31);
                        const int v0s = __shfl_sync(0xFFFFFFFFu, v0, src & 31);
                        bool hit = false;
                        if (lane < 30 && src < 32 && ((kbs >> lane_q) & 1u)) {
                            const Tet q = gather_tet<true>(p, make_int4(v0s, v0s + lane_a1, v0s + lane_a12, v0s + a123));
                            LocalBox B;
                            hit = p.pow2 ? local_box<true>(p, g, q, B) : local_box<false>(p, g, q, B);
                        }
                        const unsigned bal = __ballot_sync(0xFFFFFFFFu, hit);
                        VOX_CHECK(wq_n + __popc(bal) <= 64, CK_K4_QUEUE);
                        if (hit) wq[wq_n + __popc(bal & ((1u << lane) - 1u))] = ((u32)v0s << 3) | (u32)lane_q;
                        wq_n += __popc(bal);
                        if (wq_n >= 32) { ++grp; break; }
                    }
                } else {
                    grp = 7;
                }
                if (grp >= 7) { grp = 0; chunk += NW; }
            }
            __syncwarp();
            const int take = min(32, wq_n);
            if (!__syncthreads_or(take > 0)) break;  // (also the barrier that frees rec and s_incl)
            n = NT;
            int* r = rec + rec_off(tid);
            bool drawn = false;
            u32 carry = 0;
            if (lane + 32 < wq_n) carry = wq[lane + 32];
            if (lane < take) {
                const u32 e = wq[lane];
                const int v0 = (int)(e >> 3), q = (int)(e & 7u);
                const int a1 = (q < 2) ? lat_sx : (q < 4) ? lat_sy : 1;
                const int a3 = (q == 3 || q == 5) ? lat_sx : (q == 1 || q == 4) ? lat_sy : 1;
                const int4 id = make_int4(v0, v0 + a1, v0 + a123 - a3, v0 + a123);
                drawn = p.pow2 ? setup_pair<true, true>(p, g, id, r) : setup_pair<false, true>(p, g, id, r);
                if (r[6] == 0) atomicAdd(&s_large, 1u);
            } else {
                null_record(r, g.img_saddr);
            }
            nr = r[3];
            my_pairs += __popc(__ballot_sync(0xFFFFFFFFu, drawn));
            __syncwarp();
            if (lane + 32 < wq_n) wq[lane] = carry;  // the rest of the queue moves to the front
            wq_n -= take;
        }
        int incl = nr;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= o) incl += v;
        }
        s_incl[tid] = incl;
        if (lane == 31) s_wtot[warp] = incl;
        __syncthreads();
        // rows of the batch laid end to end: warp segment w covers [cum[w], cum[w+1])
        int cum[NW + 1];
        cum[0] = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) cum[w + 1] = cum[w] + s_wtot[w];
        const int total = cum[NW];
        const int R = (total + NT - 1) / NT;
        const int first = tid * R;
        int cnt = min(R, total - first);
        if (cnt > 0) {
            int w = 0, wb = 0;
#pragma unroll
            for (int k = 1; k < NW; ++k)
                if (first >= cum[k]) { w = k; wb = cum[k]; }
            const int local = first - wb;
            const int* inc = s_incl + w * 32;
            int j = 0;  // smallest j with inc[j] > local
#pragma unroll
            for (int step = 16; step; step >>= 1)
                if (inc[j + step - 1] <= local) j += step;
            int pi = w * 32 + j;
            int rr = local - (j ? inc[j - 1] : 0);
            VOX_CHECK(pi >= 0 && pi < NT && rr >= 0, CK_K4_RECIDX);
            LaneRec L;
            u32 ra = rec_saddr + 4u * (u32)rec_off(pi);
            lane_load(ra, L);
            for (;;) {
                lane_row(L, rr, img_stride, g.img_saddr, g.img_saddr + 4u * (u32)img_words);
                if (--cnt == 0) break;
                if (++rr == L.A.w) {  // next pair (every pair has at least one row)
                    ra += ((++pi & 3) == 0) ? 4u * SREC_W + 16u : 4u * SREC_W;  // rec_off: 16-byte pad after every 4th record
                    VOX_CHECK(pi < NT && ra == rec_saddr + 4u * (u32)rec_off(pi), CK_K4_RECIDX);
                    lane_load(ra, L);
                    rr = 0;
                }
            }
        }
        // large pairs of this batch (rare): one warp per pair, int64 ballot rasteriser
        const u32 nl = s_large;  // cumulative; stable between the barrier above and the next one
        if (nl != seen_large) {
            seen_large = nl;
            for (int i = warp; i < n; i += NW) {
                const int* r = rec + rec_off(i);
                if (r[6] == 0) raster_large_rec(r, img, lane, img_stride);
            }
        }
    }
    if (LATTICE && lane == 0 && my_pairs) atomicAdd(&s_pairs, my_pairs);
    __syncthreads();
    if (tid == 0 && s_large) atomicAdd(hdr + H_LARGE, s_large);
    if (LATTICE && tid == 0 && s_pairs) {  // the statistics K2 leaves in the header on the binned path
        const u32 np = s_pairs, old = atomicAdd(hdr + H_TOTAL, np);
        if (old + np < old) atomicAdd(hdr + H_TOTAL_HI, 1u);
        atomicAdd(hdr + H_NONEMPTY, 1u);
    }
    tile_epilogue<NT, SPARSE>(p, img, img_stride, b, bx, m, g.Y0, g.Z0, bits, hdr, so, tid);
}

// ------------------------------------------------------------------------------------------
// validation and probes
// ------------------------------------------------------------------------------------------
__global__ void k_validate(Params p, u32* hdr) {
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    bool bad = false;
    if (i < p.V) {
        int x = p.verts[3 * i], y = p.verts[3 * i + 1], z = p.verts[3 * i + 2];
        bad = bad || x < 0 || x > p.ex || y < 0 || y > p.ey || z < 0 || z > p.ez;
    }
    if (i < p.T && !p.lcx) {
        int4 id = p.tets[i];
        bad = bad || id.x < 0 || id.x >= p.V || id.y < 0 || id.y >= p.V || id.z < 0 || id.z >= p.V || id.w < 0 || id.w >= p.V;
    }
    if (p.off && i <= p.batch) {
        i64 o = p.off[i];
        if (i == 0) bad = bad || (o != 0);
        if (i == p.batch) bad = bad || (o != p.T);
        if (i > 0) bad = bad || (o < p.off[i - 1]);
    }
    if (bad) hdr[H_BAD] = 1;
}

// dependent-free integer streams: 8 independent chains per thread
template <int KIND>
__global__ void __launch_bounds__(256) k_probe(int iters, u32* sink) {
    u32 a0 = threadIdx.x, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    u32 b = blockIdx.x * 2654435761u + 12345u, c = b ^ 0x9E3779B9u;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (KIND == 0) {  // LOP3 only: alu pipe
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a7) : "r"(b), "r"(c));
            } else if (KIND == 1) {  // IMAD only: fma pipe
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a7) : "r"(b), "r"(c));
            } else {  // mixed: 4 LOP3 + 4 IMAD
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a0) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a1) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a2) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a3) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a4) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a5) : "r"(b), "r"(c));
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a6) : "r"(b), "r"(c));
                asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a7) : "r"(b), "r"(c));
            }
        }
    }
    u32 r = a0 ^ a1 ^ a2 ^ a3 ^ a4 ^ a5 ^ a6 ^ a7;
    if (r == 0x12345678u) sink[0] = r;  // practically never: keeps the chains alive
}

// ------------------------------------------------------------------------------------------
// host API
// ------------------------------------------------------------------------------------------
static int gcd_i(int a, int b) {
    while (b) { int t = a % b; a = b; b = t; }
    return a;
}
static int ilog2_exact(int v) {
    for (int s = 0; s < 31; ++s) if ((1 << s) == v) return s;
    return -1;
}
static int cuda_fail(vox_ctx* c, cudaError_t e, const char* where) {
    snprintf(c->err, sizeof(c->err), "%s: %s", where, cudaGetErrorString(e));
    return VOX_ECUDA;
}
#define CK(call)                                            \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
    } while (0)

static void set_tile(Params& p, int ty, int tz) {
    p.ty_log = ilog2_exact(ty);
    p.tz_log = ilog2_exact(tz);
    p.nbx = p.nx / 32;
    p.nby = (p.ny + ty - 1) / ty;
    p.nbz = (p.nz + tz - 1) / tz;
    p.NB = (u32)((i64)p.batch * p.nbx * p.nby * p.nbz);
}

// Binning tile: 32^3 bricks for big grids; thinner tiles (down to 32 x 8 x 8) while there would be fewer than
// four waves of CTAs (8 CTAs x 148 SMs each) or more than ~1024 tets per tile -- a tile's list is walked by ONE
// CTA, 128 pairs at a time, so long lists on few tiles leave SMs idle.
static void auto_tile(Params& p, i64 T) {
    int ty = 32, tz = 32;
    auto tiles = [&](int a, int b) { return (i64)p.batch * (p.nx / 32) * ((p.ny + a - 1) / a) * ((p.nz + b - 1) / b); };
    // (third clause, round 2: below ~16 waves the last wave's idle SMs show -- cfg3 ran 27% of K4 with SMs idle on
    //  8192 tiles of 32x16x16 and is 17% faster on 32768 of 32x8x8 -- so keep halving while a tile still has work)
    while ((tiles(ty, tz) < 4 * 1184 || T / tiles(ty, tz) > 1024 || (tiles(ty, tz) < 16 * 1184 && T / tiles(ty, tz) > 128)) &&
           (ty > 8 || tz > 8)) {
        if (tz >= ty && tz > 8) tz >>= 1; else ty >>= 1;
    }
    while (ty < 32 && (p.ny + ty - 1) / ty > 1024) ty <<= 1;
    while (tz < 32 && (p.nz + tz - 1) / tz > 1024) tz <<= 1;
    set_tile(p, ty, tz);
}

extern "C" int vox_create(vox_ctx** out, int nx, int ny, int nz, int ex, int ey, int ez, int batch) {
    if (!out) return VOX_EINVAL;
    *out = NULL;
    if (nx <= 0 || ny <= 0 || nz <= 0 || batch < 1 || ex <= 0 || ey <= 0 || ez <= 0) return VOX_EINVAL;
    if (nx % 32) return VOX_EINVAL;
    if (ex % (2 * (i64)nx) || ey % (2 * (i64)ny) || ez % (2 * (i64)nz)) return VOX_EINVAL;
    if (ex > (1 << 20) || ey > (1 << 20) || ez > (1 << 20)) return VOX_ERANGE;
    if (nx > 32768 || ny > 32768 || nz > 32768) return VOX_ERANGE;
    vox_ctx* c = (vox_ctx*)calloc(1, sizeof(vox_ctx));
    if (!c) return VOX_EINVAL;
    Params& p = c->p;
    p.nx = nx; p.ny = ny; p.nz = nz; p.ex = ex; p.ey = ey; p.ez = ez; p.batch = batch;
    p.hx = ex / nx; p.hy = ey / ny; p.hz = ez / nz;
    p.qx = ilog2_exact(2 * p.hx); p.qy = ilog2_exact(2 * p.hy); p.qz = ilog2_exact(2 * p.hz);
    p.g = gcd_i(gcd_i(p.hx, p.hy), p.hz);
    p.g_shift = ilog2_exact(p.g);
    p.sx = p.hx / p.g; p.sy = p.hy / p.g; p.sz = p.hz / p.g;
    p.lim_x = ((1 << 30) - 1) / p.sx; p.lim_y = ((1 << 30) - 1) / p.sy; p.lim_z = ((1 << 30) - 1) / p.sz;
    p.c4x = -4 * p.sx; p.c4y = -4 * p.sy; p.c4z = -4 * p.sz;
    p.pow2 = (p.qx >= 0 && p.qy >= 0 && p.qz >= 0 && p.g_shift >= 0) ? 1 : 0;
    p.fit_vol = 24.0f / (float)p.g; p.fit_ax = 16.0f * p.sx; p.fit_ay = 16.0f * p.sy; p.fit_az = 16.0f * p.sz;
    p.wpr = nx / 32;
    auto_tile(p, 0);
    if ((i64)batch * (nx / 32) * p.nby * p.nbz > 0x7FFFFFFFll) { free(c); return VOX_ERANGE; }  // one CTA per tile: gridDim.x
    c->pairs_planned = -1;
    *out = c;
    return VOX_OK;
}

static void timing_free(vox_ctx* ctx) {
    if (ctx->tm_ev) {
        for (int i = 0; i < ctx->tm_slots * TM_EV; ++i) cudaEventDestroy(ctx->tm_ev[i]);
        free(ctx->tm_ev);
    }
    ctx->tm_ev = NULL;
    ctx->tm_slots = 0;
    ctx->tm_next = 0;
}

extern "C" void vox_destroy(vox_ctx* ctx) {
    if (!ctx) return;
    timing_free(ctx);
    free(ctx);
}

extern "C" int vox_timing_enable(vox_ctx* ctx, int slots) {
    if (!ctx || slots < 0 || slots > 65536) return VOX_EINVAL;
    timing_free(ctx);
    if (slots == 0) return VOX_OK;
    ctx->tm_ev = (cudaEvent_t*)calloc((size_t)slots * TM_EV, sizeof(cudaEvent_t));
    if (!ctx->tm_ev) return VOX_EINVAL;
    ctx->tm_slots = slots;
    for (int i = 0; i < slots * TM_EV; ++i) CK(cudaEventCreate(&ctx->tm_ev[i]));
    return VOX_OK;
}

extern "C" int vox_timing_read(vox_ctx* ctx, int run, float ms_out[5]) {
    if (!ctx || !ms_out || run < 0) return VOX_EINVAL;
    if (!ctx->tm_ev || run >= ctx->tm_next || run < ctx->tm_next - ctx->tm_slots) return VOX_ESTATE;
    cudaEvent_t* e = ctx->tm_ev + (size_t)(run % ctx->tm_slots) * TM_EV;
    for (int k = 0; k < 4; ++k) CK(cudaEventElapsedTime(ms_out + k, e[k], e[k + 1]));
    CK(cudaEventElapsedTime(ms_out + 4, e[0], e[4]));
    return VOX_OK;
}

extern "C" int vox_set_tile(vox_ctx* ctx, int ty, int tz) {
    if (!ctx) return VOX_EINVAL;
    if (ctx->have_tets) return VOX_ESTATE;
    if (ilog2_exact(ty) < 2 || ty > 32 || ilog2_exact(tz) < 2 || tz > 32) return VOX_EINVAL;
    if ((ctx->p.ny + ty - 1) / ty > 1024 || (ctx->p.nz + tz - 1) / tz > 1024) return VOX_ERANGE;
    if ((i64)ctx->p.batch * (ctx->p.nx / 32) * ((ctx->p.ny + ty - 1) / ty) * ((ctx->p.nz + tz - 1) / tz) > 0x7FFFFFFFll)
        return VOX_ERANGE;  // one CTA per tile: gridDim.x
    set_tile(ctx->p, ty, tz);
    ctx->tile_user = true;
    return VOX_OK;
}

// Which path lattice input takes.  The binning passes (K1-K3 over the implied tets, then K4 on the pair lists) are the
// default: measured on every workload of profiles/r02_workloads.md they are the faster device step (cfg4 1.54 vs 1.72
// ms, cfg3 0.69 vs 0.89, cfg5 0.56 vs 0.84) except where cells are giants of many tiles each (S1: 0.245 vs 0.222), which
// is where the default picks the fused path (K0 + K4 enumerating its own candidates) by itself.  vox_set_variant(2)
// asks for the fused path regardless (its merit is the small workspace: no range array, no pair list), variant 1
// forbids it.  Lattices beyond what k0_slabs / the candidate queue were sized for always take the binning passes.
static bool fused_possible(const Params& p) {
    return p.lcx > 0 && p.lcx <= 4096 && p.lcy <= 4096 && p.lcz <= 4096 && p.V < (1ll << 28) &&
           p.batch <= 65535;  // (k0_slabs: shared-memory z table, gridDim.z = batch; queue entries are v0 << 3 | q)
}
static bool lattice_fused(const vox_ctx* ctx) {
    const Params& p = ctx->p;
    if (!fused_possible(p) || ctx->variant == 1) return false;
    if (ctx->variant == 2) return true;
    // default: only for giant cells -- a mean cell of at least 64^3 voxels (two 32-voxel tiles per axis or more)
    return (i64)p.nx * p.ny * p.nz >= 262144ll * p.lcx * p.lcy * p.lcz;
}

extern "C" int vox_set_variant(vox_ctx* ctx, int variant) {
    // 0: default.  1: lattice input always goes through the binning passes K1-K3 like a tet array.  2: lattice input
    // takes the fused path whenever the lattice is within its limits.  No effect on explicit tets.
    if (!ctx || variant < 0 || variant > 2) return VOX_EINVAL;
    ctx->variant = variant;
    ctx->p.fused = lattice_fused(ctx) ? 1 : 0;
    return VOX_OK;
}

extern "C" int vox_path(const vox_ctx* ctx) {
    if (!ctx) return VOX_EINVAL;
    if (!ctx->have_tets) return VOX_ESTATE;
    return ctx->p.lcx == 0 ? 0 : (lattice_fused(ctx) ? 2 : 1);
}

extern "C" int vox_tets(vox_ctx* ctx, const int32_t* d_verts, int64_t V, const int32_t* d_tets, int64_t T,
                        const int64_t* d_tet_offsets) {
    if (!ctx || V < 0 || T < 0) return VOX_EINVAL;
    if (T > 0 && (!d_verts || !d_tets || V == 0)) return VOX_EINVAL;
    if (ctx->p.batch > 1 && !d_tet_offsets) return VOX_EINVAL;
    if (T > 0xFFFFFFF0ll || V > 0x7FFFFFFFll) return VOX_ERANGE;
    if (((uintptr_t)d_tets & 15) != 0) return VOX_EINVAL;  // int4 loads
    ctx->p.verts = d_verts;
    ctx->p.tets = (const int4*)d_tets;
    ctx->p.V = V;
    ctx->p.T = T;
    ctx->p.off = (ctx->p.batch > 1) ? (const i64*)d_tet_offsets : NULL;
    ctx->p.keep = NULL;
    ctx->p.lcx = ctx->p.lcy = ctx->p.lcz = 0;
    ctx->p.fused = 0;
    if (!ctx->tile_user) auto_tile(ctx->p, T);
    ctx->have_tets = true;
    ctx->pairs_planned = -1;
    return VOX_OK;
}

extern "C" int vox_lattice(vox_ctx* ctx, const int32_t* d_verts, int cx, int cy, int cz, const uint8_t* d_keep) {
    if (!ctx || cx < 1 || cy < 1 || cz < 1 || !d_verts || !d_keep) return VOX_EINVAL;
    const i64 cells = (i64)ctx->p.batch * cx * cy * cz, V = (i64)ctx->p.batch * (cx + 1) * (cy + 1) * (cz + 1);
    if (6 * cells > 0xFFFFFFF0ll || V > 0x7FFFFFFFll) return VOX_ERANGE;
    Params& p = ctx->p;
    p.verts = d_verts;
    p.tets = NULL;
    p.off = NULL;
    p.keep = d_keep;
    p.lcx = cx; p.lcy = cy; p.lcz = cz;
    p.V = V;
    p.T = 6 * cells;
    p.fused = lattice_fused(ctx) ? 1 : 0;
    // (T counts the absent tets too: a carved lattice keeps a fraction, a third is assumed for the tile choice; larger
    //  tiles also mean a thinner rim of candidate cells per tile on the fused path)
    if (!ctx->tile_user) auto_tile(p, p.T / 3);
    ctx->have_tets = true;
    ctx->pairs_planned = -1;
    return VOX_OK;
}

extern "C" size_t vox_grid_words(const vox_ctx* ctx) {
    if (!ctx) return 0;
    const Params& p = ctx->p;
    return (size_t)p.batch * p.nz * p.ny * p.wpr;
}

extern "C" size_t vox_workspace_fixed_bytes(const vox_ctx* ctx) {
    if (!ctx) return 0;
    return ws_layout(ctx->p).fixed_end;
}

extern "C" size_t vox_workspace_bytes(const vox_ctx* ctx) {
    if (!ctx) return 0;
    const Params& p = ctx->p;
    if (lattice_fused(ctx))  // header + slabs + the packed vertex copy: no counters, no range array, no pair list
        return ws_layout(p).counts + align256((size_t)p.V * 16);
    i64 pairs = ctx->pairs_planned >= 0 ? ctx->pairs_planned : 4 * p.T + (i64)p.NB;
    if (pairs < 1) pairs = 1;
    return ws_layout(p).fixed_end + align256((size_t)pairs * 4);
}

// with_list: the pair list exists (vox_run); vox_plan only counts
static int enqueue_count_scan(vox_ctx* ctx, cudaStream_t st, char* ws, cudaEvent_t* ev, bool with_list) {
    Params& p = ctx->p;
    WsLayout L = ws_layout(p);
    u32* hdr = (u32*)(ws + L.hdr);
    u32* counts = (u32*)(ws + L.counts);
    u32* cursor = (u32*)(ws + L.cursor);
    u32* big = (u32*)(ws + L.big);
    uint2* range = (uint2*)(ws + L.range);
    if (ev) CK(cudaEventRecord(ev[0], st));
    // header and counts are adjacent: one memset
    CK(cudaMemsetAsync(ws + L.hdr, 0, L.cursor - L.hdr, st));
    if (p.T > 0) {
        unsigned blocks = (unsigned)((p.T + 255) / 256);
        k1_count<<<blocks, 256, 0, st>>>(p, range, counts, hdr, big);
        count_launch();
    }
    if (ev) CK(cudaEventRecord(ev[1], st));
    k2_scan<<<1, 1024, 0, st>>>(p, range, big, (u32*)(ws + L.list), counts, cursor, hdr, with_list ? 1 : 0);
    count_launch();
    CK(cudaGetLastError());
    if (ev) CK(cudaEventRecord(ev[2], st));
    return VOX_OK;
}

extern "C" int vox_plan(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, int64_t* pairs_out) {
    if (!ctx || !d_workspace || ((uintptr_t)d_workspace & 15) != 0) return VOX_EINVAL;
    if (!ctx->have_tets) return VOX_ESTATE;
    WsLayout L = ws_layout(ctx->p);
    if (ws_bytes < L.fixed_end) return VOX_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = enqueue_count_scan(ctx, st, (char*)d_workspace, NULL, false);
    if (rc) return rc;
    u32 h[HDR_WORDS];
    CK(cudaMemcpyAsync(h, (char*)d_workspace + L.hdr, sizeof(h), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    i64 total = (i64)h[H_TOTAL] | ((i64)h[H_TOTAL_HI] << 32);
    if (total > 0xFFFFFFF0ll) return VOX_ERANGE;
    ctx->pairs_planned = total;
    if (pairs_out) *pairs_out = total;
    return VOX_OK;
}

static int run_impl(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, uint32_t* d_bits_out);

extern "C" int vox_run(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, uint32_t* d_bits_out) {
    if (!ctx || !d_workspace || !d_bits_out) return VOX_EINVAL;
    ctx->sparse = SparseOut{NULL, NULL, 0};
    return run_impl(ctx, cuda_stream, d_workspace, ws_bytes, d_bits_out);
}

extern "C" int vox_run_sparse(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes,
                              uint32_t* d_table, uint32_t* d_payload, int64_t payload_capacity_tiles) {
    if (!ctx || !d_workspace || !d_table || payload_capacity_tiles < 0) return VOX_EINVAL;
    if (payload_capacity_tiles > 0 && !d_payload) return VOX_EINVAL;
    ctx->sparse.table = d_table;
    ctx->sparse.payload = d_payload;
    ctx->sparse.cap = (u32)(payload_capacity_tiles > 0xFFFFFFF0ll ? 0xFFFFFFF0ll : payload_capacity_tiles);
    int rc = run_impl(ctx, cuda_stream, d_workspace, ws_bytes, NULL);
    ctx->sparse = SparseOut{NULL, NULL, 0};
    return rc;
}

extern "C" int vox_tile_shape(const vox_ctx* ctx, int out[5]) {
    if (!ctx || !out) return VOX_EINVAL;
    const Params& p = ctx->p;
    out[0] = 1 << p.ty_log; out[1] = 1 << p.tz_log; out[2] = p.nbx; out[3] = p.nby; out[4] = p.nbz;
    return VOX_OK;
}

extern "C" int vox_sparse_status(vox_ctx* ctx, void* cuda_stream, const void* d_workspace, int64_t out[2]) {
    if (!ctx || !d_workspace) return VOX_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    WsLayout L = ws_layout(ctx->p);
    u32 h[HDR_WORDS];
    CK(cudaMemcpyAsync(h, (const char*)d_workspace + L.hdr, sizeof(h), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (out) { out[0] = h[H_MIXED]; out[1] = h[H_FULL]; }
    return (h[H_OVERFLOW] || h[H_PAYLOAD_OVERFLOW]) ? VOX_EWORKSPACE : VOX_OK;
}

// K4's grid: one CTA per tile, 3-D when the tile counts fit gridDim.y/z (sets p.grid3 for the kernel's decode)
static dim3 k4_grid(Params& p) {
    const i64 zb = (i64)p.nbz * p.batch;
    p.grid3 = (p.nby <= 65535 && zb <= 65535) ? 1 : 0;
    return p.grid3 ? dim3((unsigned)p.nbx, (unsigned)p.nby, (unsigned)zb) : dim3(p.NB);
}

static int run_impl(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes, uint32_t* d_bits_out) {
    if (((uintptr_t)d_workspace & 15) != 0) return VOX_EINVAL;  // uint2 / uint4 accesses of the workspace arrays
    if (!ctx->have_tets) return VOX_ESTATE;
    Params& p = ctx->p;
    WsLayout L = ws_layout(p);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* ws = (char*)d_workspace;
    // per-kernel timing events are not recorded into a stream capture: a captured record would be replayed with every
    // graph launch and vox_timing_read would see events that never completed outside the graph
    cudaStreamCaptureStatus cap_status = cudaStreamCaptureStatusNone;
    if (ctx->tm_ev) CK(cudaStreamIsCapturing(st, &cap_status));
    cudaEvent_t* ev = (ctx->tm_ev && cap_status == cudaStreamCaptureStatusNone)
                          ? ctx->tm_ev + (size_t)(ctx->tm_next % ctx->tm_slots) * TM_EV : NULL;
    if (lattice_fused(ctx)) {  // K0 (vertex-plane slabs) + K4 enumerating its own candidates
        if (ws_bytes < L.counts + (size_t)p.V * 16) return VOX_EWORKSPACE;
        u32* hdr = (u32*)(ws + L.hdr);
        int* slab = (int*)(ws + L.slab);
        p.verts4 = (const int4*)(ws + L.counts);  // (the binned path's arrays are not used: their room holds the copy)
        if (ev) CK(cudaEventRecord(ev[0], st));
        CK(cudaMemsetAsync(ws + L.hdr, 0, L.counts - L.hdr, st));
        // enough CTAs for two waves: one per (x plane, chunk of y rows, mesh)
        const i64 planes = (i64)(p.lcx + 1) * p.batch;
        int chunks = (int)((2 * 148 * 4 + planes - 1) / planes);
        if (chunks > p.lcy + 1) chunks = p.lcy + 1;
        if (chunks > 65535) chunks = 65535;
        const int jchunk = (p.lcy + 1 + chunks - 1) / chunks;
        dim3 grid0((unsigned)(p.lcx + 1), (unsigned)((p.lcy + 1 + jchunk - 1) / jchunk), (unsigned)p.batch);
        k0_slabs<<<grid0, 256, 2 * (size_t)(p.lcz + 1) * 4, st>>>(p.verts, p.lcx, p.lcy, p.lcz, p.ex, p.ey, p.ez, jchunk, slab,
                                                                  (int4*)(ws + L.counts));
        count_launch();
        if (ev) { CK(cudaEventRecord(ev[1], st)); CK(cudaEventRecord(ev[2], st)); CK(cudaEventRecord(ev[3], st)); }
        const SparseOut so = ctx->sparse;
        const dim3 grid4 = k4_grid(p);
        if (so.table) k4_flat<128, 8, true, true><<<grid4, 128, 0, st>>>(p, NULL, NULL, d_bits_out, hdr, so, slab);
        else k4_flat<128, 8, false, true><<<grid4, 128, 0, st>>>(p, NULL, NULL, d_bits_out, hdr, so, slab);
        count_launch();
        CK(cudaGetLastError());
        if (ev) {
            CK(cudaEventRecord(ev[4], st));
            ctx->tm_next++;
        }
        return VOX_OK;
    }
    p.verts4 = NULL;
    if (ws_bytes < L.fixed_end + 4) return VOX_EWORKSPACE;
    size_t cap = (ws_bytes - L.list) / 4;
    p.cap = (u32)(cap > 0xFFFFFFF0ull ? 0xFFFFFFF0ull : cap);
    int rc = enqueue_count_scan(ctx, st, ws, ev, true);
    if (rc) return rc;
    u32* hdr = (u32*)(ws + L.hdr);
    u32* counts = (u32*)(ws + L.counts);
    u32* cursor = (u32*)(ws + L.cursor);
    uint2* range = (uint2*)(ws + L.range);
    u32* list = (u32*)(ws + L.list);
    if (p.T > 0) {
        unsigned blocks = (unsigned)((p.T + 255) / 256);
        k3_scatter<<<blocks, 256, 0, st>>>(p, range, cursor, list, hdr);
        count_launch();
    }
    if (ev) CK(cudaEventRecord(ev[3], st));
    const SparseOut so = ctx->sparse;
    const dim3 grid4 = k4_grid(p);
    if (so.table) {
        k4_flat<128, 8, true, false><<<grid4, 128, 0, st>>>(p, counts, list, d_bits_out, hdr, so, NULL);
        count_launch();
    } else {
        k4_flat<128, 8, false, false><<<grid4, 128, 0, st>>>(p, counts, list, d_bits_out, hdr, so, NULL);  // 64 regs, 32 warps/SM
        count_launch();
    }
    CK(cudaGetLastError());
    if (ev) {
        CK(cudaEventRecord(ev[4], st));
        ctx->tm_next++;
    }
    return VOX_OK;
}

extern "C" int vox_status(vox_ctx* ctx, void* cuda_stream, const void* d_workspace, int64_t stats_out[4]) {
    if (!ctx || !d_workspace) return VOX_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    WsLayout L = ws_layout(ctx->p);
    u32 h[HDR_WORDS];
    CK(cudaMemcpyAsync(h, (const char*)d_workspace + L.hdr, sizeof(h), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (stats_out) {
        stats_out[0] = (i64)h[H_TOTAL] | ((i64)h[H_TOTAL_HI] << 32);
        stats_out[1] = h[H_CULLED];
        stats_out[2] = h[H_LARGE];
        stats_out[3] = h[H_NONEMPTY];
    }
    return h[H_OVERFLOW] ? VOX_EWORKSPACE : VOX_OK;
}

// ------------------------------------------------------------------------------------------
// vox_run_noalloc: the hot path on a workspace the library itself carries (include/vox.h)
// ------------------------------------------------------------------------------------------
// For callers that cannot obtain device memory at all (everything is owned by the host application's pool), must not
// trigger the device-wide synchronisation an allocation implies, or share the process with a global-mode graph
// capture in which cudaMalloc is an error.  The workspace is this array: part of the library's image on every
// device that loads it, never freed.  On the HOST side the name g_noalloc_scratch is only a handle for the runtime
// (a host shadow of the symbol), NOT a device address: handing it to a kernel would fault, or on a machine where the
// GPU can reach host memory quietly scribble over the wrong bytes.  The device address comes from
// cudaGetSymbolAddress, asked once per device with that device current, and is what the kernels get.
static __device__ __align__(256) unsigned char g_noalloc_scratch[VOX_NOALLOC_SCRATCH_BYTES];
enum { NOALLOC_MAX_DEVICES = 64 };
static void* g_noalloc_addr[NOALLOC_MAX_DEVICES];  // per device: address of the array there, NULL = not asked yet
static pthread_mutex_t g_noalloc_lock = PTHREAD_MUTEX_INITIALIZER;

// First call on a device: look the array's address up (this is also what makes the runtime load the library's
// device image there, so it belongs before any stream capture).  Later calls: a table read.
static int noalloc_scratch(vox_ctx* ctx, char** out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) {
        snprintf(ctx->err, sizeof(ctx->err), "vox_run_noalloc: device ordinal %d is beyond the %d this build keeps an address for",
                 dev, (int)NOALLOC_MAX_DEVICES);
        return VOX_ERANGE;
    }
    pthread_mutex_lock(&g_noalloc_lock);
    void* a = g_noalloc_addr[dev];
    cudaError_t e = cudaSuccess;
    if (!a) {
        e = cudaGetSymbolAddress(&a, g_noalloc_scratch);
        if (e == cudaSuccess && a) g_noalloc_addr[dev] = a;
    }
    pthread_mutex_unlock(&g_noalloc_lock);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    if (!a) {
        snprintf(ctx->err, sizeof(ctx->err), "vox_run_noalloc: the runtime returned no address for the built-in scratch");
        return VOX_ECUDA;
    }
    *out = (char*)a;
    return VOX_OK;
}

extern "C" int vox_run_noalloc(vox_ctx* ctx, void* cuda_stream, uint32_t* d_bits_out, int64_t stats_out[4]) {
    if (!ctx || !d_bits_out) return VOX_EINVAL;
    if (!ctx->have_tets) return VOX_ESTATE;
    // the size test comes first and touches no CUDA call: an oversized job is refused even where there is no device
    const size_t need = vox_workspace_bytes(ctx);
    if (need > (size_t)VOX_NOALLOC_SCRATCH_BYTES) {
        snprintf(ctx->err, sizeof(ctx->err),
                 "vox_run_noalloc: this mesh and grid need a %zu-byte workspace, the built-in scratch has %u "
                 "(VOX_NOALLOC_SCRATCH_BYTES); use vox_run with a workspace of your own",
                 need, (unsigned)VOX_NOALLOC_SCRATCH_BYTES);
        return VOX_EWORKSPACE;
    }
    char* scratch = NULL;
    int rc = noalloc_scratch(ctx, &scratch);
    if (rc) return rc;
    // The array still holds whatever the previous call (of any context) left.  run_impl starts by clearing the header,
    // the slab bounds and the tile counters on the stream (one cudaMemsetAsync, no allocation); the cursors, the range
    // array and the pair list are fully rewritten by K2 / K1 / K3 before they are read, so nothing else needs zeroing.
    // The whole array is handed over: the pair list gets all the room behind the fixed part.
    ctx->sparse = SparseOut{NULL, NULL, 0};
    rc = run_impl(ctx, cuda_stream, scratch, (size_t)VOX_NOALLOC_SCRATCH_BYTES, d_bits_out);
    if (rc || !stats_out) return rc;
    return vox_status(ctx, cuda_stream, scratch, stats_out);  // waits for the stream; VOX_EWORKSPACE if pairs were dropped
}

extern "C" int vox_validate(vox_ctx* ctx, void* cuda_stream, void* d_workspace, size_t ws_bytes) {
    if (!ctx || !d_workspace || ((uintptr_t)d_workspace & 15) != 0) return VOX_EINVAL;
    if (!ctx->have_tets) return VOX_ESTATE;
    Params& p = ctx->p;
    WsLayout L = ws_layout(p);
    if (ws_bytes < L.fixed_end) return VOX_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    u32* hdr = (u32*)((char*)d_workspace + L.hdr);
    CK(cudaMemsetAsync(hdr, 0, HDR_WORDS * 4, st));
    i64 n = p.V > p.T ? p.V : p.T;
    if (n < p.batch + 1) n = p.batch + 1;
    k_validate<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, hdr);
    count_launch();
    CK(cudaGetLastError());
    u32 h[HDR_WORDS];
    CK(cudaMemcpyAsync(h, hdr, sizeof(h), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return h[H_BAD] ? VOX_EDATA : VOX_OK;
}

struct ArenaLayout {
    size_t verts, tets, off, bits, ws, end;
};
static ArenaLayout arena_layout(const vox_ctx* ctx, i64 V, i64 T, size_t ws_bytes) {
    ArenaLayout A;
    size_t o = 0;
    A.verts = o; o = align256(o + (size_t)(V > 0 ? V : 1) * 12);
    A.tets = o;  o = align256(o + (size_t)(T > 0 ? T : 1) * 16);
    A.off = o;   o = align256(o + ((size_t)ctx->p.batch + 1) * 8);
    A.bits = o;  o = align256(o + vox_grid_words(ctx) * 4);
    A.ws = o;    o = o + ws_bytes;
    A.end = o;
    return A;
}

extern "C" size_t vox_host_arena_bytes(const vox_ctx* ctx, int64_t V, int64_t T) {
    if (!ctx) return 0;
    vox_ctx tmp = *ctx;
    tmp.p.T = T;
    tmp.pairs_planned = -1;
    if (!tmp.tile_user) auto_tile(tmp.p, T);  // the tile vox_tets will pick for this T
    return arena_layout(ctx, V, T, vox_workspace_bytes(&tmp)).end;
}

extern "C" int vox_run_host(vox_ctx* ctx, void* cuda_stream, const int32_t* h_verts, int64_t V, const int32_t* h_tets,
                            int64_t T, const int64_t* h_tet_offsets, void* d_arena, size_t arena_bytes,
                            uint32_t* h_bits_out) {
    if (!ctx || !d_arena || !h_bits_out || V < 0 || T < 0) return VOX_EINVAL;
    if (T > 0 && (!h_verts || !h_tets)) return VOX_EINVAL;
    if (ctx->p.batch > 1 && !h_tet_offsets) return VOX_EINVAL;
    ArenaLayout A = arena_layout(ctx, V, T, 0);
    if (arena_bytes < A.ws + 4096) return VOX_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* a = (char*)d_arena;
    if (V > 0) CK(cudaMemcpyAsync(a + A.verts, h_verts, (size_t)V * 12, cudaMemcpyHostToDevice, st));
    if (T > 0) CK(cudaMemcpyAsync(a + A.tets, h_tets, (size_t)T * 16, cudaMemcpyHostToDevice, st));
    if (ctx->p.batch > 1)
        CK(cudaMemcpyAsync(a + A.off, h_tet_offsets, ((size_t)ctx->p.batch + 1) * 8, cudaMemcpyHostToDevice, st));
    int rc = vox_tets(ctx, (const int32_t*)(a + A.verts), V, (const int32_t*)(a + A.tets), T, (const int64_t*)(a + A.off));
    if (rc) return rc;
    rc = vox_run(ctx, st, a + A.ws, arena_bytes - A.ws, (uint32_t*)(a + A.bits));
    if (rc) return rc;
    CK(cudaMemcpyAsync(h_bits_out, a + A.bits, vox_grid_words(ctx) * 4, cudaMemcpyDeviceToHost, st));
    return vox_status(ctx, st, a + A.ws, NULL);
}

// ------------------------------------------------------------------------------------------
// occupancy: k^3 sub-samples per voxel folded from the k-times finer bit grid (include/vox.h).  HBM bound:
// one thread reads the k*k fine words above one run of 32/k coarse voxels and writes 32/k bytes.
// ------------------------------------------------------------------------------------------
template <int K, int VEC>  // VEC fine words per thread and row (4: one 16-byte load per row)
__global__ void __launch_bounds__(256) k_occupancy(const u32* __restrict__ fine, int nx, int ny, int nz, int batch,
                                                   unsigned char* __restrict__ out) {
    constexpr int PER = 32 / K;                 // coarse voxels per fine word
    const int fw = (nx * K) >> 5;               // fine words per fine row
    const int fv = fw / VEC;
    const i64 total = (i64)batch * nz * ny * fv;
    const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int w = (int)(i % fv) * VEC;
    i64 rest = i / fv;
    const int y = (int)(rest % ny);
    rest /= ny;
    const int z = (int)(rest % nz);
    const i64 m = rest / nz;
    // SWAR: per fine word, K-bit group counts; even/odd groups accumulate in separate fields wide enough for K*K rows
    u32 A[VEC], B[VEC];
#pragma unroll
    for (int c = 0; c < VEC; ++c) A[c] = B[c] = 0;
    const i64 fny = (i64)ny * K, fnz = (i64)nz * K;
#pragma unroll
    for (int dz = 0; dz < K; ++dz)
#pragma unroll
        for (int dy = 0; dy < K; ++dy) {
            const u32* src = fine + ((m * fnz + (i64)z * K + dz) * fny + (i64)y * K + dy) * fw + w;
            u32 v[VEC];
            if (VEC == 4) {
                const uint4 q = __ldg(reinterpret_cast<const uint4*>(src));
                v[0] = q.x; v[1 % VEC] = q.y; v[2 % VEC] = q.z; v[3 % VEC] = q.w;
            } else {
                v[0] = __ldg(src);
            }
#pragma unroll
            for (int c = 0; c < VEC; ++c) {
                if (K == 2) {
                    const u32 s2 = (v[c] & 0x55555555u) + ((v[c] >> 1) & 0x55555555u);  // 16 fields of 2 bits: 0..2
                    A[c] += s2 & 0x33333333u;         // even voxels, 4-bit fields (sum <= 8)
                    B[c] += (s2 >> 2) & 0x33333333u;  // odd voxels
                } else {
                    const u32 s4 = v[c] - ((v[c] >> 1) & 0x77777777u) - ((v[c] >> 2) & 0x33333333u) - ((v[c] >> 3) & 0x11111111u);
                    A[c] += s4 & 0x0F0F0F0Fu;         // even voxels, byte fields (sum <= 64)
                    B[c] += (s4 >> 4) & 0x0F0F0F0Fu;  // odd voxels
                }
            }
        }
    unsigned char* dst = out + ((m * nz + z) * (i64)ny + y) * nx + (i64)w * PER;
#pragma unroll
    for (int c = 0; c < VEC; ++c) {
        if (K == 2) {
            u32 o[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {  // voxels 4q..4q+3 = A[2q], B[2q], A[2q+1], B[2q+1] (4-bit fields)
                const u32 a8 = (A[c] >> (8 * q)) & 0xFFu, b8 = (B[c] >> (8 * q)) & 0xFFu;
                o[q] = (a8 & 0xFu) | ((a8 & 0xF0u) << 12) | ((b8 & 0xFu) << 8) | ((b8 & 0xF0u) << 20);
            }
            *reinterpret_cast<uint4*>(dst + c * PER) = make_uint4(o[0], o[1], o[2], o[3]);
        } else {
            // voxels 0..7 = A0,B0,A1,B1 | A2,B2,A3,B3 (byte fields)
            *reinterpret_cast<uint2*>(dst + c * PER) = make_uint2(__byte_perm(A[c], B[c], 0x5140), __byte_perm(A[c], B[c], 0x7362));
        }
    }
}

extern "C" int vox_occupancy(void* cuda_stream, const uint32_t* d_bits_fine, int nx, int ny, int nz, int batch, int k,
                             uint8_t* d_counts_out) {
    if (!d_bits_fine || !d_counts_out || nx <= 0 || ny <= 0 || nz <= 0 || batch < 1) return VOX_EINVAL;
    if ((k != 2 && k != 4) || ((i64)nx * k) % 32 != 0) return VOX_EINVAL;
    if (((uintptr_t)d_counts_out & 15) != 0) return VOX_EINVAL;  // vector stores
    const int fw = (nx * k) >> 5;
    const bool vec = (fw % 4 == 0) && (((uintptr_t)d_bits_fine & 15) == 0);
    const i64 total = (i64)batch * nz * ny * (vec ? fw / 4 : fw);
    if (total > 0x7FFFFFFFll * 256) return VOX_ERANGE;
    const unsigned blocks = (unsigned)((total + 255) / 256);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (k == 2 && vec) k_occupancy<2, 4><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else if (k == 2) k_occupancy<2, 1><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else if (vec) k_occupancy<4, 4><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    else k_occupancy<4, 1><<<blocks, 256, 0, st>>>(d_bits_fine, nx, ny, nz, batch, d_counts_out), count_launch();
    return cudaGetLastError() == cudaSuccess ? VOX_OK : VOX_ECUDA;
}

// ------------------------------------------------------------------------------------------
// vox_pipe: transfer-overlapped pipeline over a stream of host meshes (include/vox.h)
// ------------------------------------------------------------------------------------------
enum { PIPE_MAX_DEPTH = 8 };
struct PipeSlot {
    vox_ctx* ctx;
    cudaEvent_t in_done, run_done, out_done;
    u32* h_hdr;      // pinned, HDR_WORDS
    i64 ticket;      // ticket in flight in this slot, -1 = free
    char* base;      // slice of the arena
};
struct vox_pipe {
    int depth;
    i64 maxV, maxT;
    i64 reserve_pairs;   // > 0: pair-list capacity per slot asked for by vox_pipe_reserve_pairs
    i64 next_ticket;
    cudaStream_t s_in, s_run, s_out;
    PipeSlot slot[PIPE_MAX_DEPTH];
    ArenaLayout A;       // layout of one slice (workspace last)
    size_t slice_bytes;
    bool bound;
    char err[256];
};

static int pipe_fail(vox_pipe* q, cudaError_t e, const char* where) {
    snprintf(q->err, sizeof(q->err), "%s: %s", where, cudaGetErrorString(e));
    return VOX_ECUDA;
}
#define PCK(call)                                                \
    do {                                                         \
        cudaError_t e_ = (call);                                 \
        if (e_ != cudaSuccess) return pipe_fail(pipe, e_, #call); \
    } while (0)

static void pipe_layout(vox_pipe* q) {
    vox_ctx tmp = *q->slot[0].ctx;
    tmp.p.T = q->maxT;
    tmp.pairs_planned = q->reserve_pairs > 0 ? q->reserve_pairs : -1;
    // the workspace of a slice must serve whichever path a submitted mesh takes: the binned layout (sized here from
    // max_T and the pair reservation) or, for lattice input on the fused path, header + vertex-plane slabs + the 16-byte
    // vertex copy.  Lattice dims are not known yet; (cx+1) + (cy+1) + (cz+1) <= V + 2 per mesh bounds the slabs.
    size_t ws = vox_workspace_bytes(&tmp);
    const size_t fused_ws = align256(HDR_WORDS * 4) + align256(8 * ((size_t)q->maxV + 2 * (size_t)tmp.p.batch)) +
                            align256(16 * (size_t)q->maxV);
    if (fused_ws > ws) ws = fused_ws;
    q->A = arena_layout(&tmp, q->maxV, q->maxT, ws);
    q->slice_bytes = align256(q->A.end);
}

extern "C" void vox_pipe_destroy(vox_pipe* pipe) {
    if (!pipe) return;
    if (pipe->s_out) cudaStreamSynchronize(pipe->s_out);
    if (pipe->s_run) cudaStreamSynchronize(pipe->s_run);
    if (pipe->s_in) cudaStreamSynchronize(pipe->s_in);
    for (int i = 0; i < pipe->depth; ++i) {
        PipeSlot& s = pipe->slot[i];
        if (s.in_done) cudaEventDestroy(s.in_done);
        if (s.run_done) cudaEventDestroy(s.run_done);
        if (s.out_done) cudaEventDestroy(s.out_done);
        if (s.h_hdr) cudaFreeHost(s.h_hdr);
        vox_destroy(s.ctx);
    }
    if (pipe->s_in) cudaStreamDestroy(pipe->s_in);
    if (pipe->s_run) cudaStreamDestroy(pipe->s_run);
    if (pipe->s_out) cudaStreamDestroy(pipe->s_out);
    free(pipe);
}

extern "C" int vox_pipe_create(vox_pipe** out, int nx, int ny, int nz, int ex, int ey, int ez, int batch, int depth,
                               int64_t max_V, int64_t max_T) {
    if (!out) return VOX_EINVAL;
    *out = NULL;
    if (depth < 1 || depth > PIPE_MAX_DEPTH || max_V < 0 || max_T < 0) return VOX_EINVAL;
    if (max_T > 0xFFFFFFF0ll || max_V > 0x7FFFFFFFll) return VOX_ERANGE;
    vox_pipe* pipe = (vox_pipe*)calloc(1, sizeof(vox_pipe));
    if (!pipe) return VOX_EINVAL;
    pipe->depth = depth;
    pipe->maxV = max_V;
    pipe->maxT = max_T;
    for (int i = 0; i < depth; ++i) {
        int rc = vox_create(&pipe->slot[i].ctx, nx, ny, nz, ex, ey, ez, batch);
        if (rc) { vox_pipe_destroy(pipe); return rc; }
        auto_tile(pipe->slot[i].ctx->p, max_T);  // one tile shape for every submit (the sparse table depends on it)
        pipe->slot[i].ctx->tile_user = true;
        pipe->slot[i].ticket = -1;
    }
    bool ok = cudaStreamCreateWithFlags(&pipe->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&pipe->s_run, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&pipe->s_out, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; ok && i < depth; ++i) {
        PipeSlot& s = pipe->slot[i];
        ok = cudaEventCreateWithFlags(&s.in_done, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.run_done, cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&s.out_done, cudaEventDisableTiming) == cudaSuccess &&
             cudaHostAlloc((void**)&s.h_hdr, HDR_WORDS * 4, cudaHostAllocDefault) == cudaSuccess;
    }
    if (!ok) { cudaGetLastError(); vox_pipe_destroy(pipe); return VOX_ECUDA; }
    pipe_layout(pipe);
    *out = pipe;
    return VOX_OK;
}

extern "C" int vox_pipe_set_variant(vox_pipe* pipe, int variant) {
    if (!pipe) return VOX_EINVAL;
    for (int i = 0; i < pipe->depth; ++i) {
        int rc = vox_set_variant(pipe->slot[i].ctx, variant);
        if (rc) return rc;
    }
    return VOX_OK;
}

extern "C" int vox_pipe_set_tile(vox_pipe* pipe, int ty, int tz) {
    if (!pipe) return VOX_EINVAL;
    if (pipe->bound) return VOX_ESTATE;
    for (int i = 0; i < pipe->depth; ++i) {
        int rc = vox_set_tile(pipe->slot[i].ctx, ty, tz);
        if (rc) return rc;
    }
    pipe_layout(pipe);
    return VOX_OK;
}

extern "C" int vox_pipe_reserve_pairs(vox_pipe* pipe, int64_t max_pairs) {
    if (!pipe || max_pairs < 0 || max_pairs > 0xFFFFFFF0ll) return VOX_EINVAL;
    if (pipe->bound) return VOX_ESTATE;
    pipe->reserve_pairs = max_pairs;
    pipe_layout(pipe);
    return VOX_OK;
}

extern "C" size_t vox_pipe_arena_bytes(const vox_pipe* pipe) {
    return pipe ? pipe->slice_bytes * (size_t)pipe->depth : 0;
}

extern "C" int vox_pipe_bind(vox_pipe* pipe, void* d_arena, size_t arena_bytes) {
    if (!pipe || !d_arena) return VOX_EINVAL;
    if (((uintptr_t)d_arena & 255) != 0) return VOX_EINVAL;
    if (arena_bytes < vox_pipe_arena_bytes(pipe)) return VOX_EWORKSPACE;
    for (int i = 0; i < pipe->depth; ++i) {
        if (pipe->slot[i].ticket >= 0) return VOX_ESTATE;
        pipe->slot[i].base = (char*)d_arena + (size_t)i * pipe->slice_bytes;
    }
    pipe->bound = true;
    return VOX_OK;
}

static int pipe_finish_slot(vox_pipe* pipe, PipeSlot& s, int64_t stats_out[6]) {
    PCK(cudaEventSynchronize(s.out_done));
    s.ticket = -1;
    const u32* h = s.h_hdr;
    if (stats_out) {
        stats_out[0] = (i64)h[H_TOTAL] | ((i64)h[H_TOTAL_HI] << 32);
        stats_out[1] = h[H_CULLED];
        stats_out[2] = h[H_LARGE];
        stats_out[3] = h[H_NONEMPTY];
        stats_out[4] = h[H_MIXED];
        stats_out[5] = h[H_FULL];
    }
    return (h[H_OVERFLOW] || h[H_PAYLOAD_OVERFLOW]) ? VOX_EWORKSPACE : VOX_OK;
}

struct LatticeIn { int cx, cy, cz; const uint8_t* h_keep; };  // cx == 0: explicit tets
static int pipe_submit(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets, int64_t T,
                       const int64_t* h_tet_offsets, LatticeIn lat, uint32_t* h_bits_out, uint32_t* h_payload,
                       int64_t cap_tiles, int64_t* ticket_out);

extern "C" int vox_pipe_submit(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets, int64_t T,
                               const int64_t* h_tet_offsets, uint32_t* h_bits_out, int64_t* ticket_out) {
    return pipe_submit(pipe, h_verts, V, h_tets, T, h_tet_offsets, LatticeIn{0, 0, 0, NULL}, h_bits_out, NULL, -1,
                       ticket_out);
}

extern "C" int vox_pipe_submit_sparse(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets,
                                      int64_t T, const int64_t* h_tet_offsets, uint32_t* h_table,
                                      uint32_t* h_payload, int64_t payload_capacity_tiles, int64_t* ticket_out) {
    if (payload_capacity_tiles < 0 || (payload_capacity_tiles > 0 && !h_payload)) return VOX_EINVAL;
    return pipe_submit(pipe, h_verts, V, h_tets, T, h_tet_offsets, LatticeIn{0, 0, 0, NULL}, h_table, h_payload,
                       payload_capacity_tiles, ticket_out);
}

extern "C" int vox_pipe_submit_lattice(vox_pipe* pipe, const int32_t* h_verts, int cx, int cy, int cz,
                                       const uint8_t* h_keep, uint32_t* h_out, uint32_t* h_payload,
                                       int64_t payload_capacity_tiles, int64_t* ticket_out) {
    if (cx < 1 || cy < 1 || cz < 1 || !h_keep || !h_verts) return VOX_EINVAL;
    if (payload_capacity_tiles > 0 && !h_payload) return VOX_EINVAL;
    if (!pipe) return VOX_EINVAL;
    const int64_t batch = pipe->slot[0].ctx->p.batch;
    const int64_t cells = batch * cx * cy * cz;
    return pipe_submit(pipe, h_verts, batch * (cx + 1) * (cy + 1) * (cz + 1), NULL, 6 * cells, NULL,
                       LatticeIn{cx, cy, cz, h_keep}, h_out, h_payload, payload_capacity_tiles < 0 ? -1 : payload_capacity_tiles,
                       ticket_out);
}

// cap_tiles < 0: dense (h_bits_out = grid); else sparse (h_bits_out = tile table, h_payload host-mapped)
static int pipe_submit(vox_pipe* pipe, const int32_t* h_verts, int64_t V, const int32_t* h_tets, int64_t T,
                       const int64_t* h_tet_offsets, LatticeIn lat, uint32_t* h_bits_out, uint32_t* h_payload,
                       int64_t cap_tiles, int64_t* ticket_out) {
    if (!pipe || !h_bits_out || V < 0 || T < 0) return VOX_EINVAL;
    if (!pipe->bound) return VOX_ESTATE;
    if (V > pipe->maxV || T > pipe->maxT) return VOX_ERANGE;
    if (T > 0 && (!h_verts || (!h_tets && !lat.cx))) return VOX_EINVAL;
    PipeSlot& s = pipe->slot[pipe->next_ticket % pipe->depth];
    vox_ctx* ctx = s.ctx;
    if (ctx->p.batch > 1 && !h_tet_offsets && !lat.cx) return VOX_EINVAL;
    if (s.ticket >= 0) {  // slot still in flight and never waited on: its result is complete but unclaimed
        PCK(cudaEventSynchronize(s.out_done));
        s.ticket = -1;
    }
    const ArenaLayout& A = pipe->A;
    char* a = s.base;
    // everything that can be refused is checked BEFORE the first enqueue: the mesh binding (host-side state only)
    // and the device view of the caller's payload buffer
    int rc = lat.cx ? vox_lattice(ctx, (const int32_t*)(a + A.verts), lat.cx, lat.cy, lat.cz, (const uint8_t*)(a + A.tets))
                    : vox_tets(ctx, (const int32_t*)(a + A.verts), V, (const int32_t*)(a + A.tets), T,
                               (const int64_t*)(a + A.off));
    if (rc) return rc;
    void* d_payload = NULL;
    if (cap_tiles > 0) PCK(cudaHostGetDevicePointer(&d_payload, h_payload, 0));
    // From here on work is in flight on the slot's arena slice: a failure must not return before it has drained
    // (the next submit would pick the same slot and overwrite the slice under the running copies / kernels).
#define PCK_DRAIN(call)                                            \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) {                                   \
            pipe_fail(pipe, e_, #call);                            \
            cudaStreamSynchronize(pipe->s_in);                     \
            cudaStreamSynchronize(pipe->s_run);                    \
            cudaStreamSynchronize(pipe->s_out);                    \
            return VOX_ECUDA;                                      \
        }                                                          \
    } while (0)
    // copy-in stream
    if (V > 0) PCK_DRAIN(cudaMemcpyAsync(a + A.verts, h_verts, (size_t)V * 12, cudaMemcpyHostToDevice, pipe->s_in));
    if (lat.cx)  // the keep mask (one byte per cell) travels in the slot's tet region
        PCK_DRAIN(cudaMemcpyAsync(a + A.tets, lat.h_keep, (size_t)(T / 6), cudaMemcpyHostToDevice, pipe->s_in));
    else if (T > 0) PCK_DRAIN(cudaMemcpyAsync(a + A.tets, h_tets, (size_t)T * 16, cudaMemcpyHostToDevice, pipe->s_in));
    if (ctx->p.batch > 1 && !lat.cx)
        PCK_DRAIN(cudaMemcpyAsync(a + A.off, h_tet_offsets, ((size_t)ctx->p.batch + 1) * 8, cudaMemcpyHostToDevice, pipe->s_in));
    PCK_DRAIN(cudaEventRecord(s.in_done, pipe->s_in));
    // compute stream
    PCK_DRAIN(cudaStreamWaitEvent(pipe->s_run, s.in_done, 0));
    size_t out_bytes = vox_grid_words(ctx) * 4;
    if (cap_tiles < 0) {
        rc = vox_run(ctx, pipe->s_run, a + A.ws, pipe->slice_bytes - A.ws, (uint32_t*)(a + A.bits));
    } else {
        // the kernel stores mixed tiles straight into the caller's pinned payload buffer (device view of it)
        rc = vox_run_sparse(ctx, pipe->s_run, a + A.ws, pipe->slice_bytes - A.ws, (uint32_t*)(a + A.bits),
                            (uint32_t*)d_payload, cap_tiles);
        out_bytes = (size_t)ctx->p.NB * 4;  // the tile table lives where the dense grid would
    }
    if (rc) {
        if (rc == VOX_ECUDA) snprintf(pipe->err, sizeof(pipe->err), "%s", ctx->err);
        cudaStreamSynchronize(pipe->s_in);
        cudaStreamSynchronize(pipe->s_run);
        return rc;
    }
    PCK_DRAIN(cudaEventRecord(s.run_done, pipe->s_run));
    // copy-out stream
    PCK_DRAIN(cudaStreamWaitEvent(pipe->s_out, s.run_done, 0));
    PCK_DRAIN(cudaMemcpyAsync(h_bits_out, a + A.bits, out_bytes, cudaMemcpyDeviceToHost, pipe->s_out));
    PCK_DRAIN(cudaMemcpyAsync(s.h_hdr, a + A.ws + ws_layout(ctx->p).hdr, HDR_WORDS * 4, cudaMemcpyDeviceToHost, pipe->s_out));
    PCK_DRAIN(cudaEventRecord(s.out_done, pipe->s_out));
#undef PCK_DRAIN
    s.ticket = pipe->next_ticket++;
    if (ticket_out) *ticket_out = s.ticket;
    return VOX_OK;
}

extern "C" int vox_pipe_wait(vox_pipe* pipe, int64_t ticket, int64_t stats_out[6]) {
    if (!pipe || ticket < 0) return VOX_EINVAL;
    PipeSlot& s = pipe->slot[ticket % pipe->depth];
    if (s.ticket != ticket) return VOX_ESTATE;  // never submitted, already waited on, or overwritten
    return pipe_finish_slot(pipe, s, stats_out);
}

extern "C" int vox_pipe_tile_shape(const vox_pipe* pipe, int out[5]) {
    return pipe ? vox_tile_shape(pipe->slot[0].ctx, out) : VOX_EINVAL;
}

extern "C" const char* vox_pipe_last_error(const vox_pipe* pipe) { return pipe ? pipe->err : ""; }

extern "C" int vox_probe_int32(void* cuda_stream, int kind, int blocks, int iters, uint32_t* d_sink, double* ops_out) {
    if (blocks <= 0 || iters <= 0 || !d_sink) return VOX_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (kind == 0) k_probe<0><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    else if (kind == 1) k_probe<1><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    else k_probe<2><<<blocks, 256, 0, st>>>(iters, d_sink), count_launch();
    if (cudaGetLastError() != cudaSuccess) return VOX_ECUDA;
    if (ops_out) *ops_out = (double)blocks * 256.0 * (double)iters * 64.0;
    return VOX_OK;
}

extern "C" uint64_t vox_kernel_launches(void) { return __atomic_load_n(&g_launches, __ATOMIC_RELAXED); }

extern "C" int vox_debug_check_status(uint32_t* code_out) {
#ifdef VOX_CHECKS
    unsigned int c = 0, zero = 0;
    if (cudaDeviceSynchronize() != cudaSuccess) return VOX_ECUDA;
    if (cudaMemcpyFromSymbol(&c, g_check, sizeof(c)) != cudaSuccess) return VOX_ECUDA;
    if (cudaMemcpyToSymbol(g_check, &zero, sizeof(zero)) != cudaSuccess) return VOX_ECUDA;
    if (code_out) *code_out = c;
    return 1;
#else
    if (code_out) *code_out = 0;
    return 0;
#endif
}

// Operand-level self-test of the integer helpers of the row walk (checked build only; include/vox.h).  One thread per
// element; the helpers are the very functions K4 inlines.
#ifdef VOX_CHECKS
__global__ void __launch_bounds__(256) k_selftest(int op, const i64* __restrict__ a, const i64* __restrict__ b, i64 n,
                                                  int* __restrict__ out) {
    const i64 i = (i64)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const i64 x = a[i], y = b[i];
    int r = 0;
    if (op == 0) r = span_bound((int)x, -(int)(u32)y, recip_up((u32)y));
    else if (op == 1) r = span_bound((int)x, -(int)(u32)y, (int)(0xFFFFFFFFu / (u32)y + 1u));
    else if (op == 2) r = (int)(((u32)x * (u32)div_magic((int)y)) >> 16);
    else if (op == 3) r = span64_bound(x, y);
    else if (op == 4) r = recip_up((u32)y);
    out[i] = r;
}
#endif
extern "C" int vox_debug_selftest(void* cuda_stream, int op, const int64_t* d_a, const int64_t* d_b, int64_t n,
                                  int32_t* d_out) {
#ifdef VOX_CHECKS
    if (op < 0 || op > 4 || n < 0 || (n > 0 && (!d_a || !d_b || !d_out))) return VOX_EINVAL;
    if (n == 0) return 1;
    k_selftest<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(op, (const i64*)d_a, (const i64*)d_b, n, d_out);
    count_launch();
    return cudaGetLastError() == cudaSuccess ? 1 : VOX_ECUDA;
#else
    (void)cuda_stream; (void)op; (void)d_a; (void)d_b; (void)n; (void)d_out;
    return 0;
#endif
}

extern "C" const char* vox_strerror(int code) {
    switch (code) {
        case VOX_OK: return "ok";
        case VOX_EINVAL: return "invalid argument";
        case VOX_ERANGE: return "argument out of the supported range";
        case VOX_EWORKSPACE: return "workspace too small";
        case VOX_ECUDA: return "CUDA runtime error (see vox_last_error)";
        case VOX_ESTATE: return "call order violated";
        case VOX_EDATA: return "mesh data out of range";
        default: return "unknown error";
    }
}

extern "C" const char* vox_last_error(const vox_ctx* ctx) { return ctx ? ctx->err : ""; }
