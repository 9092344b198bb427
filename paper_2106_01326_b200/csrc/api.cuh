// api.cuh -- part of vox.cu (included there, once): host side of the C ABI: create/tets/lattice/plan/run/status/noalloc/validate/run_host.
#pragma once

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
