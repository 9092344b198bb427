// common.cuh -- part of vox.cu (included there, once): host context (Params, vox_ctx, workspace layout), check macros and the integer-geometry device helpers.
#pragma once

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
