// pipe.cuh -- part of vox.cu (included there, once): vox_pipe_*: the transfer-overlapped pipeline.
#pragma once

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
